// rflbm_host.cuh — host-side handle and the step-kernel launch/dispatch templates, shared by rflbm.cu (the C-ABI)
// and rflbm_step_inst.cu (which instantiates the step kernels, one (precision, phase) pair per translation unit so
// that the ~190 kernel instantiations compile in parallel; build.py).
#pragma once
#include <cuda_runtime.h>

#include "../../include/rflbm.h"
#include "rflbm_kernels.cuh"
#include "rflbm_step_tma.cuh"

using namespace rflbm_dev;

struct rflbm {
    int nx, ny, nz;
    long long N;
    long long QS;        // elements between population arrays inside a buffer: N rounded up to 32 plus padding
    double tau, kT, rho0;
    uint64_t seed;
    int precision;
    int walls;
    int model;           // RFLBM_MODEL_REG / RFLBM_MODEL_BGK
    double tau_g;        // ghost relaxation time 1/omega_g (1 = the paper's final scheme)
    int scheme;          // RFLBM_SCHEME_AB (two buffers) / RFLBM_SCHEME_AA (one buffer, in place)
    int aa_phase;        // AA: 0 = natural layout (next step is the in-place one), 1 = after an in-place step
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
    CUtensorMap tmap[2];  // TMA descriptors of the two population buffers (fp64, nx >= 128, nx even)
    bool tma_ok;
    int variant;          // RFLBM_KERNEL_AUTO / _PLAIN / _TMA
    int tma_rows;         // y rows walked by one block of the TMA kernel
    char err[512];
};


template <typename real, bool WALLS, bool FORCE, bool NOISE, bool BGK, bool GHOST, int PHASE>
static inline void launch_one(rflbm* h, const StepParams<real>& P, bool tma)
{
    // A-B: read buf[cur], write the other buffer; AA: one buffer, in place
    const real* src = (const real*)h->buf[h->cur];
    real* dst = (real*)h->buf[PHASE == STEP_AB ? (h->cur ^ 1) : h->cur];
    if (tma) {
        const dim3 grid((h->nx + TILE_X - 1) / TILE_X, (h->ny + h->tma_rows - 1) / h->tma_rows, h->nz);
        step_kernel_tma<real, WALLS, FORCE, NOISE, BGK, GHOST, PHASE><<<grid, TILE_X, 0, h->stream>>>(
            h->tmap[h->cur], src, dst, P, h->tma_rows);
    } else {
        step_kernel<real, WALLS, FORCE, NOISE, BGK, GHOST, PHASE><<<h->grid, h->block, 0, h->stream>>>(src, dst, P);
    }
}

// variant bits: 16 = general ghost rate, 8 = BGK-FLBM, 4 = walls, 2 = force, 1 = noise
// (BGK and the ghost rate carry no force and exclude each other: rflbm_set_model / set_ghost_tau / set_force)
template <typename real, int PHASE>
void dispatch_variant(rflbm* h, const StepParams<real>& P, int variant, bool tma)
{
    switch (variant) {
        case 0: launch_one<real, false, false, false, false, false, PHASE>(h, P, tma); break;
        case 1: launch_one<real, false, false, true, false, false, PHASE>(h, P, tma); break;
        case 2: launch_one<real, false, true, false, false, false, PHASE>(h, P, tma); break;
        case 3: launch_one<real, false, true, true, false, false, PHASE>(h, P, tma); break;
        case 4: launch_one<real, true, false, false, false, false, PHASE>(h, P, tma); break;
        case 5: launch_one<real, true, false, true, false, false, PHASE>(h, P, tma); break;
        case 6: launch_one<real, true, true, false, false, false, PHASE>(h, P, tma); break;
        case 7: launch_one<real, true, true, true, false, false, PHASE>(h, P, tma); break;
        case 8: launch_one<real, false, false, false, true, false, PHASE>(h, P, tma); break;
        case 9: launch_one<real, false, false, true, true, false, PHASE>(h, P, tma); break;
        case 12: launch_one<real, true, false, false, true, false, PHASE>(h, P, tma); break;
        case 13: launch_one<real, true, false, true, true, false, PHASE>(h, P, tma); break;
        case 16: launch_one<real, false, false, false, false, true, PHASE>(h, P, tma); break;
        case 17: launch_one<real, false, false, true, false, true, PHASE>(h, P, tma); break;
        case 20: launch_one<real, true, false, false, false, true, PHASE>(h, P, tma); break;
        default: launch_one<real, true, false, true, false, true, PHASE>(h, P, tma); break;    // 21
    }
}

