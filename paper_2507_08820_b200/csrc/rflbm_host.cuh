// rflbm_host.cuh — host-side handle and the step-kernel launch/dispatch templates, shared by rflbm.cu (the C-ABI)
// and rflbm_step_inst.cu (which instantiates the step kernels, one (precision, phase) pair per translation unit so
// that the kernel instantiations compile in parallel; build.py).
#pragma once
#include <cuda_runtime.h>

#include "../../include/rflbm.h"
#include "rflbm_kernels.cuh"
#include "rflbm_step_tma.cuh"

using namespace rflbm_dev;

struct rflbm {
    int nx, ny, nz;      // owned lattice
    long long N;         // nx*ny*nz
    int px;              // row pitch of the internal buffers (elements): nx rounded up so that rows are 16-byte aligned
    int slab;            // 1 after rflbm_set_slab: ghost layers below and above, global z for walls and the RNG key
    int z0, nzg;         // slab: global z of the first owned layer, global number of layers
    long long QS;        // slot stride of the internal buffers = px (layout P[z][y][q][x])
    double tau, kT, rho0;
    uint64_t seed;
    int precision;
    int walls;
    int model;           // RFLBM_MODEL_REG / RFLBM_MODEL_BGK
    double tau_g;        // ghost relaxation time 1/omega_g (1 = the paper's final scheme)
    int scheme;          // RFLBM_SCHEME_AB (two buffers) / RFLBM_SCHEME_AA (one buffer, in place)
    int aa_phase;        // AA: 0 = natural layout (next step is the in-place one), 1 = after an in-place step
    int halo_mode;       // slab: what the next halo exchange carries (HALO_NONE / HALO_FILL / HALO_HOME, rflbm.cu)
    int halo_done;       // slab: bit 0 / bit 1 = rflbm_halo_unpack(LOW / HIGH) done since the last step
    double g[3];
    bool force;
    void* ws;            // borrowed workspace
    size_t ws_bytes;
    void* buf[2];        // population buffers inside ws (AA: buf[1] is NULL)
    double* acc;         // 4 KiB reduction scratch inside ws
    f64x2* tables;       // 12 KiB Box-Muller tables inside ws (uploaded by set_workspace)
    int cur;             // buffer holding P_{t-1}
    bool inited;
    uint64_t t;
    uint64_t launches;
    cudaStream_t stream;
    dim3 block, grid;
    CUtensorMap tmap[2];  // TMA descriptors of the two population buffers (load boxes: TX + halo, 3 populations)
    CUtensorMap tmap_out[2];  // the same buffers with the store box of one warp: 32 x, all 27 populations of one row
    bool tma_ok;
    int tma_tx;           // tile width of the TMA kernel for this lattice: 128, 64 or 32 (0: nx < 32, plain kernel only)
    int variant;          // RFLBM_KERNEL_AUTO / _PLAIN / _TMA
    int tma_rows;         // y rows walked by one block of the TMA kernel
    const char* last_kernel;   // what the last rflbm_step launched (static string)
    int zc, zn;           // owned layers [zc, zc+zn) the next launch covers (0, nz except inside rflbm_run_host's pipeline)
    cudaStream_t copy_stream;  // optional second stream for the copies of rflbm_run_host (rflbm_set_copy_stream)
    int inject_fail;           // test hook (rflbm_debug_inject_failure): the n-th checked CUDA call of the next pipelined job fails
    char err[512];
};

inline Geom make_geom(const rflbm* h)
{
    Geom G;
    G.nx = h->nx; G.ny = h->ny; G.nz = h->nz;
    G.nzs = h->nz + (h->slab ? 2 : 0);
    G.z_lo = h->slab ? 1 : 0;
    G.zc = h->zc;
    G.zg0 = h->slab ? h->z0 - 1 : 0;
    G.nzg = h->slab ? h->nzg : h->nz;
    G.px = Q * h->px;                              // P[z][y][q][x]: consecutive rows of one population are 27 px apart
    G.pxy = (long long)Q * h->px * h->ny;
    G.QS = h->px;
    G.N = h->N;
    return G;
}

// TX = 0: the plain one-thread-per-site kernel; TX = 128 / 64 / 32: the TMA-staged kernel with that tile width
template <typename real, int TX, bool WALLS, bool FORCE, bool NOISE, bool BGK, bool GHOST, int PHASE>
static inline void launch_one(rflbm* h, const StepParams<real>& P)
{
    // A-B: read buf[cur], write the other buffer; AA: one buffer, in place
    const real* src = (const real*)h->buf[h->cur];
    real* dst = (real*)h->buf[PHASE == STEP_AB ? (h->cur ^ 1) : h->cur];
    if constexpr (TX != 0) {
        const dim3 grid((h->nx + TX - 1) / TX, (h->ny + h->tma_rows - 1) / h->tma_rows, h->zn);
        auto kern = step_kernel_tma<real, TX, WALLS, FORCE, NOISE, BGK, GHOST, PHASE>;
        constexpr int dyn = tma_store_bytes<real, PHASE>();       // per-warp output boxes of the TMA-store instantiations
        kern<<<grid, BLOCK_T, dyn, h->stream>>>(h->tmap[h->cur], h->tmap_out[PHASE == STEP_AB ? (h->cur ^ 1) : h->cur], src, dst, P,
                                                 h->tma_rows);
    } else {
        const dim3 grid(h->grid.x, h->grid.y, h->zn);
        step_kernel<real, WALLS, FORCE, NOISE, BGK, GHOST, PHASE><<<grid, h->block, 0, h->stream>>>(src, dst, P);
    }
}

// variant bits: 16 = general ghost rate, 8 = BGK-FLBM, 4 = walls, 2 = force, 1 = noise
// (BGK and the ghost rate carry no force and exclude each other: rflbm_set_model / set_ghost_tau / set_force)
template <typename real, int PHASE, int TX>
void dispatch_variant(rflbm* h, const StepParams<real>& P, int variant)
{
    switch (variant) {
        case 0: launch_one<real, TX, false, false, false, false, false, PHASE>(h, P); break;
        case 1: launch_one<real, TX, false, false, true, false, false, PHASE>(h, P); break;
        case 2: launch_one<real, TX, false, true, false, false, false, PHASE>(h, P); break;
        case 3: launch_one<real, TX, false, true, true, false, false, PHASE>(h, P); break;
        case 4: launch_one<real, TX, true, false, false, false, false, PHASE>(h, P); break;
        case 5: launch_one<real, TX, true, false, true, false, false, PHASE>(h, P); break;
        case 6: launch_one<real, TX, true, true, false, false, false, PHASE>(h, P); break;
        case 7: launch_one<real, TX, true, true, true, false, false, PHASE>(h, P); break;
        case 8: launch_one<real, TX, false, false, false, true, false, PHASE>(h, P); break;
        case 9: launch_one<real, TX, false, false, true, true, false, PHASE>(h, P); break;
        case 12: launch_one<real, TX, true, false, false, true, false, PHASE>(h, P); break;
        case 13: launch_one<real, TX, true, false, true, true, false, PHASE>(h, P); break;
        case 16: launch_one<real, TX, false, false, false, false, true, PHASE>(h, P); break;
        case 17: launch_one<real, TX, false, false, true, false, true, PHASE>(h, P); break;
        case 20: launch_one<real, TX, true, false, false, false, true, PHASE>(h, P); break;
        default: launch_one<real, TX, true, false, true, false, true, PHASE>(h, P); break;    // 21
    }
}
