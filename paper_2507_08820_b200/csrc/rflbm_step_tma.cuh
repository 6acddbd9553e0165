// rflbm_step_tma.cuh — the hot kernel, TMA-staged (sm_100a): one time step of Eq.24 on an fp64 or fp32 lattice with
// any nx >= 32 (tiles of 128, 64 or 32 sites; the internal row pitch is padded to whole 128-byte lines).
//
// Why (profiles/r01a_*): in the plain one-thread-per-site kernel every one of the 27 neighbour loads costs 4-5
// integer instructions of per-thread 64-bit address arithmetic, and a block's memory latency is exposed between
// its load phase and its ~1300-instruction compute phase.  Here a tile is 128 consecutive x of one row; the 27
// row segments it needs arrive as NINE `cp.async.bulk.tensor` copies (box = 132 x, 1 y, 1 z, 3 populations: the
// three q = 3b+9c+{0,1,2} that share the source row (y-cy, z-cz)), issued by one elected thread of warp 0 into
// shared memory.  The TMA unit generates the addresses, applies the y/z shift and the periodic wrap in y and z
// (and fetches the opposite populations 26-q at the site itself for halfway bounce-back, R12); the copy of row
// y+1 is issued as soon as row y has been moved from shared memory to registers, so it overlaps the whole
// collision of row y.  Threads read their 27 populations with LDS [tid*8 + immediate].  A block walks `rows`
// consecutive y rows, so the Box-Muller tables are staged once per block.
//
// TMA needs 16-byte aligned box starts, so a box starts at the even x0-2 and spans 132 elements; the thread at
// x reads element tid+3 (cx=-1, source x+1), tid+2 (cx=0) or tid+1 (cx=+1, source x-1) of its row.
// The one thing TMA cannot do is the periodic wrap in x (out-of-bounds box elements are zero-filled): the two
// threads at x = 0 and x = nx-1 load their 9 wrapped populations directly from global memory, issued before the
// mbarrier wait so that the latency hides behind it.
//
// Variants that were measured and dropped (512^3, kT=1e-4): one private 32-site pipeline per
// warp (no block barrier, but 4x the TMA issue work and 12 % more L2->SM traffic: no faster); a persistent grid
// with static or ticket-based strip assignment (1.1-1.5x SLOWER: warps of a block drift apart, the 16-byte halos
// of neighbouring tiles stop hitting in L2).
#pragma once
#include <cuda.h>

#include "rflbm_kernels.cuh"

namespace rflbm_dev {

constexpr int BLOCK_T = 128;                  // threads per block
constexpr int BOX_Q = 3;                      // populations per box
constexpr int TMA_MIN_NX = 32;
// Tile = TX consecutive x of RB = 128/TX consecutive rows (TX = 128, 64 or 32: every lattice with nx >= 32 takes this
// kernel).  Per element type: 16-byte halo on each side of a row segment (2 doubles / 4 floats),
// box = [x0-HALO, x0+TX+HALO) x 3 populations.
template <typename real, int TX> struct TmaGeom {
    static constexpr int HALO = 16 / (int)sizeof(real);
    static constexpr int RB = BLOCK_T / TX;                                          // rows per block step
    static constexpr int BOX_X = TX + 2 * HALO;                                      // 132 doubles / 136 floats at TX = 128
    static constexpr int BOX_BYTES = BOX_X * BOX_Q * (int)sizeof(real);              // 3168 B / 1632 B per copy
    static constexpr int BOX_PITCH_BYTES = (BOX_BYTES + 127) / 128 * 128;            // destinations stay 128-byte aligned
    static constexpr int BOX_PITCH = BOX_PITCH_BYTES / (int)sizeof(real);            // in elements
    static constexpr int ROW_STAGE = 9 * BOX_PITCH;                                  // elements per staged row
    static constexpr int STAGE_BYTES = RB * 9 * BOX_PITCH_BYTES;                     // 28.8 KB / 15.0 KB at TX = 128
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
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
__device__ __forceinline__ void tma_load_box(uint32_t dst, const CUtensorMap* tmap, int x, int y, int z, int q, uint32_t bar)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
        ::"r"(dst), "l"((unsigned long long)tmap), "r"(x), "r"(q), "r"(y), "r"(z), "r"(bar)      // tensor map dimensions: (x, q, y, z)
        : "memory");
}

// store of one box from shared memory (bulk async-group completion); same coordinate order as the loads
__device__ __forceinline__ void tma_store_box(const CUtensorMap* tmap, uint32_t src, int x, int y, int z, int q)
{
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group [%0, {%1, %2, %3, %4}], [%5];"
                 ::"l"((unsigned long long)tmap), "r"(x), "r"(q), "r"(y), "r"(z), "r"(src)
                 : "memory");
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}
__device__ __forceinline__ void tma_store_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

__device__ __forceinline__ bool elect_one()
{
    uint32_t pred;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "elect.sync _|p, 0xffffffff;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(pred));
    return pred != 0;
}

// issue the 9 box copies of one row segment (x0, y, z) of the tile; one thread.  The caller has armed the mbarrier.
// PHASE (rflbm_kernels.cuh): STEP_AB pulls slot q of the neighbour row (bounce-back: slot 26-q of the own row);
// STEP_AA_EVEN reads slot q of the own row; STEP_AA_ODD pulls slot 26-q of the neighbour row (bounce-back: slot q of
// the own row).  A box holds three consecutive slots, so "26-q" boxes start at 24-3b-9c and hold the rows reversed.
template <typename real, int TX, bool WALLS, int PHASE>
__device__ __forceinline__ void issue_row(const CUtensorMap* tmap, uint32_t s_in, uint32_t bar, int x0, int y, int z,
                                          int zg, const Geom& G)
{
    using T = TmaGeom<real, TX>;
    const int ys[3] = {(y + 1 == G.ny) ? 0 : y + 1, y, (y == 0) ? G.ny - 1 : y - 1};     // y - cy, index b = cy + 1
    const int zs[3] = {(z + 1 == G.nzs) ? 0 : z + 1, z, (z == 0) ? G.nzs - 1 : z - 1};   // slab mode: never wraps
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        // with walls the fluid layers are zg = 1..nzg-2; x - c_q is solid iff (cz=+1 and zg==1) or (cz=-1 and zg==nzg-2):
        // the population comes back from the site itself as 26-q; the three q' = 26-q of a box are 24-3b-9c + {0,1,2}
        const bool bounce = WALLS && ((c == 2 && zg == 1) || (c == 0 && zg == G.nzg - 2));
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const uint32_t dst = s_in + (uint32_t)((3 * c + b) * T::BOX_PITCH_BYTES);
            const int q_fwd = 3 * b + 9 * c, q_rev = 24 - 3 * b - 9 * c;
            if (PHASE == STEP_AA_EVEN) tma_load_box(dst, tmap, x0 - T::HALO, y, z, q_fwd, bar);
            else if (WALLS && bounce) tma_load_box(dst, tmap, x0 - T::HALO, y, z, PHASE == STEP_AB ? q_rev : q_fwd, bar);
            else tma_load_box(dst, tmap, x0 - T::HALO, ys[b], zs[c], PHASE == STEP_AB ? q_fwd : q_rev, bar);
        }
    }
}

// the RB rows yb .. yb+RB-1 (those below y_end) of the tile
template <typename real, int TX, bool WALLS, int PHASE>
__device__ __forceinline__ void issue_tile(const CUtensorMap* tmap, uint32_t s_in, uint32_t bar, int x0, int yb, int y_end,
                                           int z, int zg, const Geom& G)
{
    using T = TmaGeom<real, TX>;
    const int nrows = min(T::RB, y_end - yb);
    mbar_expect_tx(bar, (uint32_t)nrows * 9u * (uint32_t)T::BOX_BYTES);
#pragma unroll
    for (int r = 0; r < T::RB; ++r)
        if (r < nrows)
            issue_row<real, TX, WALLS, PHASE>(tmap, s_in + (uint32_t)(r * 9 * T::BOX_PITCH_BYTES), bar, x0, yb + r, z, zg, G);
}

// Which instantiations write their results with bulk tensor STORES (SASS UTMASTG): each warp stages its 32 sites x 27
// populations in shared memory ([27][32], conflict-free STS.[tid*size + immediate]) and lane 0 issues ONE
// cp.async.bulk.tensor store of the box (32 x, 27 q, 1 y, 1 z) — in the layout P[z][y][q][x] the 27 rows a lattice row
// writes are consecutive, so one box replaces 27 STG and their 54 address instructions per warp.  No block barrier: a
// warp waits only for its own previous box to have been read (cp.async.bulk.wait_group.read) before it refills it.
// Measured in one call each, sustained, 512^3 (profiles/r02_variants.md): fp32 A-B 5.177 -> 5.044 and 5.491 -> 5.300 ms
// (-2.6 / -3.5 %, the fp32 kernel is issue bound; 6 blocks of 79 registers instead of 8 of 64: the box stage makes it 7
// by shared memory anyway); fp64 A-B 9.639 -> 9.658 and 10.272 -> 10.291 ms (+0.2 %: 39 fewer instructions per 32 sites
// and a slightly higher clock under the power cap, but the fence + warp sync at the end of every row is exposed with 3
// warps per scheduler), so fp64 keeps its per-thread streaming stores.  Issuing the box one row late, behind the next
// block barrier: fp64 +2 %, fp32 +0.6 % slower than the immediate form.  The odd AA phase cannot use a box at all (its
// cx = +-1 populations move by one element: box starts must be multiples of 16 bytes).
#ifndef RFLBM_F64_AB_BLOCKS
#define RFLBM_F64_AB_BLOCKS 3        // resident blocks per SM of the fp64 A-B instantiation (see the comment below)
#endif
template <typename real, int PHASE> __host__ __device__ constexpr bool tma_store() { return sizeof(real) == 4 && PHASE != STEP_AA_ODD; }
template <typename real, int PHASE> __host__ __device__ constexpr int tma_store_bytes()
{
    return tma_store<real, PHASE>() ? (BLOCK_T / 32) * Q * 32 * (int)sizeof(real) : 0;
}

// fp64, A-B scheme: 3 blocks per SM (up to 168 registers; 41 KB each).  Measured against 4 blocks of 128 registers in
// one call, sustained: 9.73 vs 9.80 and 9.86 vs 9.92 ms (24 fewer instructions per site, no spills; 5 blocks of 96
// registers: 10.13).  The in-place phases keep 4 blocks (10.09 vs 10.14 with 3).  fp32: 64 registers, 15 KB -> 8 blocks.
template <typename real, int TX, bool WALLS, bool FORCE, bool NOISE, bool BGK, bool GHOST, int PHASE>
__global__ void __launch_bounds__(BLOCK_T, sizeof(real) == 8 ? (PHASE == STEP_AB ? RFLBM_F64_AB_BLOCKS : 4) : (tma_store<real, PHASE>() ? 6 : 8))
step_kernel_tma(const __grid_constant__ CUtensorMap tmap_src, const __grid_constant__ CUtensorMap tmap_dst, const real* src, real* dst,
                const __grid_constant__ StepParams<real> P, int rows)
{
    constexpr bool TSTORE = tma_store<real, PHASE>();
    extern __shared__ __align__(128) unsigned char s_dyn[];    // TSTORE: one [27][32] output box per warp
    using T = TmaGeom<real, TX>;
    constexpr bool TABLES = NOISE && sizeof(real) == 8;         // the fp32 Box-Muller needs no tables
    __shared__ __align__(128) real s_stage[T::STAGE_BYTES / sizeof(real)];
    __shared__ f64x2 s_tab[TABLES ? LOG_TABLE_N + SC_TABLE_N : 1];
    __shared__ __align__(8) unsigned long long s_bar;

    const Geom& G = P.G;
    const int z = (int)blockIdx.z + G.zc + G.z_lo, zg = z + G.zg0;
    if (WALLS && solid_layer(G, zg)) return;                   // solid layers are never updated
    const int tid = threadIdx.x;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);    // warp-uniform for the compiler too
    const int r = (T::RB == 1) ? 0 : __shfl_sync(0xffffffffu, tid / TX, 0);   // row of the tile this warp works on
    const int xl = tid - r * TX;
    const int x0 = blockIdx.x * TX;
    const int y_begin = blockIdx.y * rows;
    const int y_end = min(y_begin + rows, G.ny);
    const uint32_t bar = smem_u32(&s_bar), in0 = smem_u32(&s_stage[0]);

    if (warp == 0 && elect_one()) {
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        issue_tile<real, TX, WALLS, PHASE>(&tmap_src, in0, bar, x0, y_begin, y_end, z, zg, G);
    }
    if (TABLES) stage_tables(P.tables, s_tab);                  // ends with __syncthreads()
    else __syncthreads();                                       // mbarrier init visible to every waiter

    const int x = x0 + xl;
    const bool active = x < G.nx;
    const bool wrap_lo = (x == 0), wrap_hi = (x == G.nx - 1);
    const bool edge_warp = __any_sync(0xffffffffu, wrap_lo || wrap_hi);
    const uint32_t QS32 = (uint32_t)G.QS;                        // QS < 2^32 (rflbm_create)
    const real* tile = &s_stage[0] + r * T::ROW_STAGE + xl;
    const bool bounce_lo = WALLS && zg == 1, bounce_hi = WALLS && zg == G.nzg - 2;
    uint32_t parity = 0;
    const int lane = tid & 31;
    real* const s_out = reinterpret_cast<real*>(s_dyn) + (size_t)(tid >> 5) * (Q * 32) + lane;     // this thread's column of its warp's box
    const uint32_t out_box = smem_u32(reinterpret_cast<real*>(s_dyn) + (size_t)warp * (Q * 32));
    // row-invariant parts of the storage index and of the Philox site key (the key is < 2^32: 32-bit arithmetic is exact)
    const long long s_col = (long long)x + G.pxy * z;
    const uint32_t site_col = (uint32_t)x + (uint32_t)G.nx * (uint32_t)G.ny * (uint32_t)zg;

    for (int yb = y_begin; yb < y_end; yb += T::RB) {
        const int y = yb + r;
        const bool row_ok = (T::RB == 1) || y < y_end;          // warp-uniform
        const long long s = s_col + (long long)G.px * y;
        // periodic wrap in x: TMA zero-fills these 9 values; fetch them early, use them after the barrier
        real wv[3][3];
        if (PHASE != STEP_AA_EVEN && edge_warp && row_ok) {     // warp-uniform branch: interior warps skip all of this
            if (wrap_lo || wrap_hi) {
                const int ysr[3] = {(y + 1 == G.ny) ? 0 : y + 1, y, (y == 0) ? G.ny - 1 : y - 1};
                const int zsr[3] = {(z + 1 == G.nzs) ? 0 : z + 1, z, (z == 0) ? G.nzs - 1 : z - 1};
#pragma unroll
                for (int c = 0; c < 3; ++c)
#pragma unroll
                    for (int b = 0; b < 3; ++b) {
                        const long long row = (long long)G.px * ysr[b] + G.pxy * zsr[c];
                        // x+1 -> 0 for cx = -1 (a = 0); x-1 -> nx-1 for cx = +1 (a = 2); nx >= 32 here
                        const int qa = (wrap_hi ? 0 : 2) + 3 * b + 9 * c;
                        const int slot = (PHASE == STEP_AB) ? qa : 26 - qa;
                        const long long at = (long long)slot * G.QS + row + (wrap_hi ? 0 : G.nx - 1);
                        wv[c][b] = (PHASE == STEP_AB) ? __ldg(src + at) : src[at];   // AA: the buffer is written in place
                    }
            }
        }
        mbar_wait(bar, parity);
        parity ^= 1u;
        real g[3][3][3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const bool bounce = (c == 2 && bounce_lo) || (c == 0 && bounce_hi);
#pragma unroll
            for (int b = 0; b < 3; ++b) {
                const real* box = tile + (3 * c + b) * T::BOX_PITCH;
                // forward boxes hold slots q in rows a = 0,1,2; reversed boxes hold q' = 26-q in ascending q': row 2-a.
                // Pulled rows are read with the x shift -cx, local ones (bounce-back, even AA phase) at xl+HALO.
                const bool local = (PHASE == STEP_AA_EVEN) || (WALLS && bounce);
                const bool reversed = (PHASE == STEP_AB) ? (WALLS && bounce) : (PHASE == STEP_AA_ODD && !(WALLS && bounce));
                if (local && reversed) {
                    g[c][b][0] = box[2 * T::BOX_X + T::HALO];
                    g[c][b][1] = box[1 * T::BOX_X + T::HALO];
                    g[c][b][2] = box[0 * T::BOX_X + T::HALO];
                } else if (local) {
                    g[c][b][0] = box[0 * T::BOX_X + T::HALO];
                    g[c][b][1] = box[1 * T::BOX_X + T::HALO];
                    g[c][b][2] = box[2 * T::BOX_X + T::HALO];
                } else if (reversed) {
                    g[c][b][0] = box[2 * T::BOX_X + T::HALO + 1];
                    g[c][b][1] = box[1 * T::BOX_X + T::HALO];
                    g[c][b][2] = box[0 * T::BOX_X + T::HALO - 1];
                } else {
                    g[c][b][0] = box[0 * T::BOX_X + T::HALO + 1];
                    g[c][b][1] = box[1 * T::BOX_X + T::HALO];
                    g[c][b][2] = box[2 * T::BOX_X + T::HALO - 1];
                }
            }
        }
        __syncthreads();                                       // the tile is in registers: the stage is free
        if (warp == 0 && yb + T::RB < y_end && elect_one())
            issue_tile<real, TX, WALLS, PHASE>(&tmap_src, in0, bar, x0, yb + T::RB, y_end, z, zg, G);

        if (PHASE != STEP_AA_EVEN && edge_warp && row_ok) {
            if (wrap_lo || wrap_hi) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const bool bounce = (c == 2 && bounce_lo) || (c == 0 && bounce_hi);
                    if (WALLS && bounce) continue;             // bounced populations come from the site itself
#pragma unroll
                    for (int b = 0; b < 3; ++b) {
                        if (wrap_hi) g[c][b][0] = wv[c][b];
                        else g[c][b][2] = wv[c][b];
                    }
                }
            }
        }
        if ((TSTORE ? __any_sync(0xffffffffu, active) : active) && row_ok) {       // TSTORE: whole warps (lanes beyond nx are clipped by the store)
            const uint32_t site = site_col + (uint32_t)G.nx * (uint32_t)y;
            collide<real, FORCE, NOISE, BGK, GHOST>(g, P, site, s_tab, s_tab + LOG_TABLE_N);
            if (PHASE == STEP_AA_ODD) {
                // push to the neighbours x + c_q (slot q), misaligned by one element for cx = +-1: the partial
                // sectors at the ends of a warp's 256 bytes are completed in L2 by the neighbouring warp's store
                // Three per-thread column pointers (x-1, x, x+1 with the periodic wrap) plus a (row, slot) offset that is
                // the same for the whole block: two address instructions per store, like the aligned stores below
                // (the generic scatter() of rflbm_kernels.cuh rebuilds a 64-bit per-thread index for each of the 27).
                const long long xm = (x == 0) ? G.nx - 1 : x - 1, xp = (x + 1 == G.nx) ? 0 : x + 1;
                const unsigned long long col[3] = {reinterpret_cast<unsigned long long>(dst + xm),
                                                   reinterpret_cast<unsigned long long>(dst + x),
                                                   reinterpret_cast<unsigned long long>(dst + xp)};
                const unsigned long long own = reinterpret_cast<unsigned long long>(dst + s);
                const int yd[3] = {(y == 0) ? G.ny - 1 : y - 1, y, (y + 1 == G.ny) ? 0 : y + 1};
                const int zd[3] = {(z == 0) ? G.nzs - 1 : z - 1, z, (z + 1 == G.nzs) ? 0 : z + 1};
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    // x + c_q is solid iff (cz=-1 and zg==1) or (cz=+1 and zg==nzg-2): back to the site itself as 26-q
                    const bool bounce = WALLS && ((c == 0 && bounce_lo) || (c == 2 && bounce_hi));
#pragma unroll
                    for (int b = 0; b < 3; ++b) {
                        const long long rowoff = (long long)G.px * yd[b] + G.pxy * zd[c];      // block-uniform
#pragma unroll
                        for (int a = 0; a < 3; ++a) {
                            const int q = a + 3 * b + 9 * c;
                            const unsigned long long push = col[a] + (unsigned long long)(((long long)q * G.QS + rowoff) * (long long)sizeof(real));
                            const unsigned long long back = own + (unsigned long long)QS32 * ((unsigned)sizeof(real) * (26 - q));
                            __stcs(reinterpret_cast<real*>((WALLS && bounce) ? back : push), g[c][b][a]);
                        }
                    }
                }
            } else if (TSTORE) {
                // all stores of the warp as ONE bulk tensor store: the 27 rows of a lattice row are consecutive in P[z][y][q][x]
                if (lane == 0) tma_store_wait_read();           // the previous box has been read out of shared memory
                __syncwarp();
#pragma unroll
                for (int c = 0; c < 3; ++c)
#pragma unroll
                    for (int b = 0; b < 3; ++b)
#pragma unroll
                        for (int a = 0; a < 3; ++a) {
                            const int q = a + 3 * b + 9 * c;
                            s_out[((PHASE == STEP_AA_EVEN) ? 26 - q : q) * 32] = g[c][b][a];
                        }
                fence_proxy_async();                            // generic-proxy writes -> visible to the async proxy
                __syncwarp();
                if (lane == 0) tma_store_box(&tmap_dst, out_box, x, y, z, 0);     // lanes beyond nx are clipped by the tensor map
            } else {
                const unsigned long long out = reinterpret_cast<unsigned long long>(dst + s);
#pragma unroll
                for (int c = 0; c < 3; ++c)
#pragma unroll
                    for (int b = 0; b < 3; ++b)
#pragma unroll
                        for (int a = 0; a < 3; ++a) {
                            // out + QS * sizeof(real) * slot as a 32x32->64 product (QS < 2^32): one IMAD.WIDE.U32 with the addend folded in.
                            // (An inline `mad.wide.u32` came out of ptxas as IMAD.WIDE + IADD3 + IMAD.X: 3 instructions.)
                            const int q = a + 3 * b + 9 * c;
                            const unsigned slot = (PHASE == STEP_AA_EVEN) ? 26 - q : q;
                            const unsigned long long at = out + (unsigned long long)QS32 * ((unsigned)sizeof(real) * slot);
                            __stcs(reinterpret_cast<real*>(at), g[c][b][a]);
                        }
            }
        }
    }
    if (TSTORE && lane == 0) tma_store_wait_read();             // shared memory stays valid until the last box has been read
}

}  // namespace rflbm_dev
