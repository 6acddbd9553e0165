// rflbm.cu — C-ABI library (include/rflbm.h) over the kernels in rflbm_kernels.cuh.
//
// Host side only: argument validation, parameter marshalling, launches on the caller's stream.
// The library never allocates device memory and never creates a stream (include/rflbm.h).
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "rflbm_host.cuh"

static size_t real_size(const rflbm* h) { return h->precision == RFLBM_F64 ? sizeof(double) : sizeof(float); }
static size_t pop_elems(const rflbm* h);
static size_t pop_bytes(const rflbm* h) { return pop_elems(h) * real_size(h); }
static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
static constexpr size_t TABLE_BYTES = (LOG_TABLE_N + SC_TABLE_N) * sizeof(f64x2);
enum { HALO_NONE = 0, HALO_FILL = 1, HALO_HOME = 2 };

// Storage layout: P[z][y][q][x], i.e. the 27 populations of one lattice ROW are 27 consecutive
// padded rows of px elements: slot stride QS = px, row stride 27 px, layer stride 27 px ny.  Everything a block touches
// in one row step (27 rows written, 9 source rows of 3 populations each read) then lies in a few contiguous pieces of
// 12-110 KB instead of 54 streams a gigabyte apart.
static void set_layout(rflbm* h)
{
    h->QS = h->px;
}
static size_t pop_elems(const rflbm* h) { return (size_t)Q * (size_t)h->px * (size_t)h->ny * (size_t)(h->nz + (h->slab ? 2 : 0)); }

// launch grid of the one-thread-per-site kernels over the owned layers [zc, zc+zn) of the next launch
static dim3 zgrid(const rflbm* h) { return dim3(h->grid.x, h->grid.y, (unsigned)h->zn); }

static int fail(rflbm* h, int code, const char* fmt, ...)
{
    if (h) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(h->err, sizeof(h->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

static int check_cuda(rflbm* h, cudaError_t e, const char* what)
{
    if (e == cudaSuccess) return RFLBM_OK;
    return fail(h, RFLBM_ECUDA, "%s: %s", what, cudaGetErrorString(e));
}

static int after_launch(rflbm* h, const char* what)
{
    h->launches++;
    return check_cuda(h, cudaPeekAtLastError(), what);
}

// cuTensorMapEncodeTiled through the runtime's driver entry point: libcuda is not linked, so the library still
// loads on a machine without a driver (the CPU-side ABI tests).
typedef CUresult (*encode_tiled_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// L2 promotion of the tensor maps, per precision (compile-time).  NONE: measured against L2_256B (rounds 1-2) and L2_128B
// in one call at 512^3, sustained (profiles/r03_variants.md): fp64 9.69 -> 9.64-9.65 ms, fp32 4.986 -> 4.981 ms, fp32
// L2 read sectors -10 %, DRAM reads 1.053 -> 1.036 x algorithmic (a box is 16 bytes wider than its tile on either side;
// promotion turned those two half sectors into two 256-byte fetches).
#ifndef RFLBM_TMAP_PROMO_F64
#define RFLBM_TMAP_PROMO_F64 CU_TENSOR_MAP_L2_PROMOTION_NONE
#endif
#ifndef RFLBM_TMAP_PROMO_F32
#define RFLBM_TMAP_PROMO_F32 CU_TENSOR_MAP_L2_PROMOTION_NONE
#endif

// 4-D view [nzs][ny][27][nx] (x pitch px) of one population buffer, box = BOX_X consecutive x of BOX_Q populations of one row
static bool make_tensor_map(rflbm* h, void* base, CUtensorMap* out, bool store_box = false)
{
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
        qres != cudaDriverEntryPointSuccess) {
        cudaGetLastError();
        return false;
    }
    const bool f64 = h->precision == RFLBM_F64;
    const cuuint64_t es = f64 ? 8 : 4;
    // dimensions (x, q, y, z): strides px, 27 px, 27 px ny elements (each a multiple of the one before)
    const cuuint64_t dims[4] = {(cuuint64_t)h->nx, (cuuint64_t)Q, (cuuint64_t)h->ny, (cuuint64_t)(h->nz + (h->slab ? 2 : 0))};
    const cuuint64_t strides[3] = {(cuuint64_t)h->px * es, (cuuint64_t)Q * h->px * es, (cuuint64_t)Q * h->px * h->ny * es};
    const cuuint32_t box[4] = {store_box ? 32u : (cuuint32_t)(h->tma_tx + 2 * (16 / (int)es)), store_box ? (cuuint32_t)Q : (cuuint32_t)BOX_Q, 1, 1};     // 16-byte aligned starts
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    const CUresult r = ((encode_tiled_fn)fn)(out, f64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, base, dims, strides, box, estr,
                                             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                             f64 ? RFLBM_TMAP_PROMO_F64 : RFLBM_TMAP_PROMO_F32, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

extern "C" int rflbm_create(int nx, int ny, int nz, double tau, double kT, double rho0, uint64_t seed, int precision,
                            rflbm_t** out)
{
    if (!out) return RFLBM_EINVAL;
    *out = nullptr;
    if (nx < 1 || ny < 1 || nz < 1) return RFLBM_EINVAL;
    if ((double)nx * (double)ny * (double)nz >= 4294967296.0) return RFLBM_EINVAL;
    // Geom::px = 27 x the padded row length (nx rounded up by at most 31 elements) is an int in every kernel
    if (nx > RFLBM_MAX_NX) return RFLBM_EINVAL;
    if (!std::isfinite(tau) || !(tau > 0.5)) return RFLBM_EINVAL;
    if (!std::isfinite(kT) || kT < 0.0) return RFLBM_EINVAL;
    if (!std::isfinite(rho0) || !(rho0 > 0.0)) return RFLBM_EINVAL;
    if (precision != RFLBM_F64 && precision != RFLBM_F32) return RFLBM_EINVAL;
    // one thread per site; a warp covers 32 consecutive x whenever nx >= 32
    int bx = 8;
    while (bx < nx && bx < 128) bx *= 2;
    const int by = 128 / bx;
    // gridDim.y / gridDim.z limits of the one-thread-per-site kernels (the TMA grid has fewer blocks in y)
    if ((ny + by - 1) / by > 65535 || nz > 65535) return RFLBM_EINVAL;
    rflbm* h = new (std::nothrow) rflbm;
    if (!h) return RFLBM_ENOMEM;
    memset(h, 0, sizeof(*h));
    h->nx = nx; h->ny = ny; h->nz = nz;
    h->N = (long long)nx * ny * nz;
    h->tau_g = 1.0;
    h->tau = tau; h->kT = kT; h->rho0 = rho0; h->seed = seed; h->precision = precision;
    // internal row pitch: whole 128-byte lines per row, so that every lattice with nx >= 32 can take the TMA kernel
    // (16-byte aligned box starts) and every warp's stores are line aligned; tiny lattices stay packed
    const int line = 128 / (int)real_size(h);
    h->px = (nx >= TMA_MIN_NX) ? (nx + line - 1) / line * line : nx;
    // tile width of the TMA kernel: the one that wastes the fewest threads on the ragged last tile, the widest on a tie
    h->tma_tx = 0;
    if (nx >= TMA_MIN_NX) {
        long long best = -1;
        for (int tx = 128; tx >= 32; tx /= 2) {
            const long long covered = (long long)((nx + tx - 1) / tx) * tx;
            if (best < 0 || covered < best) { best = covered; h->tma_tx = tx; }
        }
    }
    set_layout(h);
    if ((double)h->QS >= 4294967296.0) { delete h; return RFLBM_EINVAL; }
    h->nzg = nz;
    h->block = dim3(bx, by, 1);
    h->grid = dim3((nx + bx - 1) / bx, (ny + by - 1) / by, nz);
    h->tma_rows = 16;
    h->last_kernel = "";
    h->zc = 0; h->zn = nz;
    *out = h;
    return RFLBM_OK;
}

extern "C" size_t rflbm_workspace_bytes(const rflbm_t* h)
{
    if (!h) return 0;
    return (h->scheme == RFLBM_SCHEME_AA ? 1 : 2) * align_up(pop_bytes(h), 256) + 4096 + TABLE_BYTES;
}

extern "C" int rflbm_set_workspace(rflbm_t* h, void* dev_ptr, size_t bytes)
{
    if (!h) return RFLBM_EINVAL;
    if (!dev_ptr) return fail(h, RFLBM_EINVAL, "workspace pointer is NULL");
    if (bytes < rflbm_workspace_bytes(h))
        return fail(h, RFLBM_ENOMEM, "workspace too small: %zu < %zu bytes", bytes, rflbm_workspace_bytes(h));
    if (((uintptr_t)dev_ptr & 255u) != 0) return fail(h, RFLBM_ENOMEM, "workspace must be 256-byte aligned");
    h->ws = dev_ptr;
    h->ws_bytes = bytes;
    const size_t pb = align_up(pop_bytes(h), 256);
    const size_t nbuf = (h->scheme == RFLBM_SCHEME_AA) ? 1 : 2;
    h->buf[0] = dev_ptr;
    h->buf[1] = (nbuf == 2) ? (char*)dev_ptr + pb : nullptr;
    h->acc = (double*)((char*)dev_ptr + nbuf * pb);
    h->tables = (f64x2*)((char*)dev_ptr + nbuf * pb + 4096);
    h->aa_phase = 0;
    h->cur = 0;
    h->inited = false;
    h->halo_mode = HALO_NONE;
    h->halo_done = 0;
    // The only device writes outside the handle's stream (include/rflbm.h says so): the scratch clear and the
    // Box-Muller tables (host-generated, long double libm), both on the legacy stream, followed by a host-side wait
    // for that stream: a pageable H2D copy may return before the DMA has landed and cudaMemset is asynchronous, and
    // the kernels that read them run on h->stream, which need not be ordered against the legacy stream.
    if (int rc0 = check_cuda(h, cudaMemset(h->acc, 0, 4096), "scratch clear")) return rc0;
    f64x2 host_tab[LOG_TABLE_N + SC_TABLE_N];                  // 12 KB on the stack: no shared state between handles
    fill_normal_tables(host_tab, host_tab + LOG_TABLE_N);
    int rc = check_cuda(h, cudaMemcpy(h->tables, host_tab, TABLE_BYTES, cudaMemcpyHostToDevice), "table upload");
    if (rc != RFLBM_OK) return rc;
    rc = check_cuda(h, cudaStreamSynchronize(0), "table upload (sync)");
    if (rc != RFLBM_OK) return rc;
    // TMA path: every lattice with nx >= 32 (rows of the internal buffers are 16-byte aligned by construction)
    h->tma_ok = false;
    if (h->tma_tx != 0)
        h->tma_ok = make_tensor_map(h, h->buf[0], &h->tmap[0]) && (nbuf == 1 || make_tensor_map(h, h->buf[1], &h->tmap[1])) &&
                    make_tensor_map(h, h->buf[0], &h->tmap_out[0], true) && (nbuf == 1 || make_tensor_map(h, h->buf[1], &h->tmap_out[1], true));
    return RFLBM_OK;
}

extern "C" int rflbm_set_stream(rflbm_t* h, void* cuda_stream)
{
    if (!h) return RFLBM_EINVAL;
    h->stream = (cudaStream_t)cuda_stream;
    return RFLBM_OK;
}

extern "C" int rflbm_set_walls_z(rflbm_t* h, int on)
{
    if (!h) return RFLBM_EINVAL;
    if (on && (h->slab ? h->nzg : h->nz) < 3) return fail(h, RFLBM_EINVAL, "walls need nz >= 3");
    if (h->inited) return fail(h, RFLBM_ESTATE, "set_walls_z must precede init/set_populations");
    h->walls = on ? 1 : 0;
    return RFLBM_OK;
}

extern "C" int rflbm_set_force(rflbm_t* h, double gx, double gy, double gz)
{
    if (!h) return RFLBM_EINVAL;
    if (!std::isfinite(gx) || !std::isfinite(gy) || !std::isfinite(gz)) return fail(h, RFLBM_EINVAL, "non-finite force");
    if ((h->model == RFLBM_MODEL_BGK || h->tau_g != 1.0) && (gx != 0.0 || gy != 0.0 || gz != 0.0))
        return fail(h, RFLBM_EINVAL, "BGK-FLBM and the general ghost rate carry no body force");
    h->g[0] = gx; h->g[1] = gy; h->g[2] = gz;
    h->force = (gx != 0.0 || gy != 0.0 || gz != 0.0);
    return RFLBM_OK;
}

template <typename real>
static FieldParams<real> field_params(const rflbm* h)
{
    FieldParams<real> P;
    P.G = make_geom(h);
    P.hgx = (real)(0.5 * h->g[0]); P.hgy = (real)(0.5 * h->g[1]); P.hgz = (real)(0.5 * h->g[2]);
    P.aa = (h->scheme == RFLBM_SCHEME_AA) ? 1 : 0;
    P.ghost_in = h->slab ? 1 : 0;
    return P;
}

template <typename real>
static StepParams<real> step_params(const rflbm* h, uint64_t t)
{
    StepParams<real> P;
    const double omega = 1.0 / h->tau;
    P.G = make_geom(h);
    P.half_omc = (real)(0.5 * (1.0 - omega));
    const double omega_g = 1.0 / h->tau_g;
    P.omc_g = (real)(1.0 - omega_g);
    // Eq.9 per unit sqrt(rho): sqrt(3 kT omega_k (2 - omega_k)) prod_axis s_p, s = (1, sqrt3/6, sqrt2/6)
    // omega_k = omega_h for k = 4..9; ghosts: 1 in Reg-FLBM (:215), the same omega in BGK-FLBM (Eq.11)
    const double nh = std::sqrt(3.0 * h->kT * omega * (2.0 - omega));
    const double ng = (h->model == RFLBM_MODEL_BGK) ? nh : std::sqrt(3.0 * h->kT * omega_g * (2.0 - omega_g));
    const double s1 = std::sqrt(3.0) / 6.0, s2 = std::sqrt(2.0) / 6.0;
    P.amp[AMP_200] = (real)(nh * s2);
    P.amp[AMP_110] = (real)(nh * s1 * s1);
    P.amp[AMP_210] = (real)(ng * s2 * s1);
    P.amp[AMP_111] = (real)(ng * s1 * s1 * s1);
    P.amp[AMP_220] = (real)(ng * s2 * s2);
    P.amp[AMP_211] = (real)(ng * s2 * s1 * s1);
    P.amp[AMP_221] = (real)(ng * s2 * s2 * s1);
    P.amp[AMP_222] = (real)(ng * s2 * s2 * s2);
    P.gx = (real)h->g[0]; P.gy = (real)h->g[1]; P.gz = (real)h->g[2];
    P.force_stress = (real)(1.0 - 0.5 * omega);
    P.rng = make_philox_step(h->seed, t);
    P.tables = h->tables;
    return P;
}

// which gather reads the observable state S_t out of the current buffer (rflbm_kernels.cuh)
static int gather_mode(const rflbm* h)
{
    return h->scheme == RFLBM_SCHEME_AB ? GATHER_AB : (h->aa_phase ? GATHER_AA1 : GATHER_AA0);
}
#define RFLBM_LAUNCH_OBSERVABLE_GRID(GRID, KERNEL, ...)                                                           \
    do {                                                                                                          \
        const int gm_ = gather_mode(h);                                                                           \
        const dim3 grid_ = (GRID);                                                                                \
        if (h->walls) {                                                                                           \
            if (gm_ == GATHER_AB) KERNEL<real, true, GATHER_AB><<<grid_, h->block, 0, h->stream>>>(__VA_ARGS__);          \
            else if (gm_ == GATHER_AA1) KERNEL<real, true, GATHER_AA1><<<grid_, h->block, 0, h->stream>>>(__VA_ARGS__);   \
            else KERNEL<real, true, GATHER_AA0><<<grid_, h->block, 0, h->stream>>>(__VA_ARGS__);                          \
        } else {                                                                                                  \
            if (gm_ == GATHER_AB) KERNEL<real, false, GATHER_AB><<<grid_, h->block, 0, h->stream>>>(__VA_ARGS__);         \
            else if (gm_ == GATHER_AA1) KERNEL<real, false, GATHER_AA1><<<grid_, h->block, 0, h->stream>>>(__VA_ARGS__);  \
            else KERNEL<real, false, GATHER_AA0><<<grid_, h->block, 0, h->stream>>>(__VA_ARGS__);                         \
        }                                                                                                         \
    } while (0)
#define RFLBM_LAUNCH_OBSERVABLE(KERNEL, ...) RFLBM_LAUNCH_OBSERVABLE_GRID(zgrid(h), KERNEL, __VA_ARGS__)

// slab mode: what the next halo exchange has to carry
//   A-B, and AA after an even step: the ghost layers must receive the neighbours' face populations before the next
//   pull (HALO_FILL); AA after an odd step: the ghost layers hold what this slab pushed across its faces and the
//   neighbours have to take it home (HALO_HOME); AA in the natural layout with nothing pushed yet: nothing.
static void after_state_change(rflbm* h)
{
    h->halo_done = 0;
    if (!h->slab) h->halo_mode = HALO_NONE;
    else if (h->scheme == RFLBM_SCHEME_AB) h->halo_mode = HALO_FILL;
    else h->halo_mode = HALO_NONE;                 // AA after init / set_populations; rflbm_step sets it afterwards
}
static bool halo_pending(const rflbm* h) { return h->slab && h->halo_mode != HALO_NONE && h->halo_done != 3; }
#define RFLBM_REQUIRE_HALO(h)                                                                                    \
    if (halo_pending(h)) return fail(h, RFLBM_ESTATE, "slab: halo exchange pending (rflbm_halo_pack / rflbm_halo_unpack on both sides)")

// ---------------------------------------------------------------- init / import / export
template <typename real>
static int do_init(rflbm* h, const void* rho, const void* u)
{
    const FieldParams<real> P = field_params<real>(h);
    if (h->walls)
        init_kernel<real, true><<<zgrid(h), h->block, 0, h->stream>>>((const real*)rho, (const real*)u, h->rho0,
                                                                      (real*)h->buf[0], (real*)h->buf[1], P);
    else
        init_kernel<real, false><<<zgrid(h), h->block, 0, h->stream>>>((const real*)rho, (const real*)u, h->rho0,
                                                                       (real*)h->buf[0], (real*)h->buf[1], P);
    return after_launch(h, "init_kernel");
}

extern "C" int rflbm_init(rflbm_t* h, const void* rho_dev, const void* u_dev)
{
    if (!h) return RFLBM_EINVAL;
    if (!h->ws) return fail(h, RFLBM_ESTATE, "rflbm_init before rflbm_set_workspace");
    if ((rho_dev == nullptr) != (u_dev == nullptr)) return fail(h, RFLBM_EINVAL, "rho and u must both be given or both NULL");
    const int rc = (h->precision == RFLBM_F64) ? do_init<double>(h, rho_dev, u_dev) : do_init<float>(h, rho_dev, u_dev);
    if (rc != RFLBM_OK) return rc;
    h->cur = 0;
    h->aa_phase = 0;
    h->t = 0;
    h->inited = true;
    after_state_change(h);
    return RFLBM_OK;
}

template <typename real>
static int do_import(rflbm* h, const void* f)
{
    const FieldParams<real> P = field_params<real>(h);
    if (h->walls)
        import_kernel<real, true><<<zgrid(h), h->block, 0, h->stream>>>((const real*)f, (real*)h->buf[0], (real*)h->buf[1], P);
    else
        import_kernel<real, false><<<zgrid(h), h->block, 0, h->stream>>>((const real*)f, (real*)h->buf[0], (real*)h->buf[1], P);
    return after_launch(h, "import_kernel");
}

extern "C" int rflbm_set_populations(rflbm_t* h, const void* f_dev, uint64_t step)
{
    if (!h) return RFLBM_EINVAL;
    if (!f_dev) return fail(h, RFLBM_EINVAL, "f_dev is NULL");
    if (!h->ws) return fail(h, RFLBM_ESTATE, "rflbm_set_populations before rflbm_set_workspace");
    const int rc = (h->precision == RFLBM_F64) ? do_import<double>(h, f_dev) : do_import<float>(h, f_dev);
    if (rc != RFLBM_OK) return rc;
    h->cur = 0;
    h->aa_phase = 0;
    h->t = step;
    h->inited = true;
    after_state_change(h);
    return RFLBM_OK;
}

template <typename real>
static int do_export(rflbm* h, void* f)
{
    const FieldParams<real> P = field_params<real>(h);
    RFLBM_LAUNCH_OBSERVABLE(export_kernel, (const real*)h->buf[h->cur], (real*)f, P);
    return after_launch(h, "export_kernel");
}

extern "C" int rflbm_get_populations(rflbm_t* h, void* f_dev)
{
    if (!h) return RFLBM_EINVAL;
    if (!f_dev) return fail(h, RFLBM_EINVAL, "f_dev is NULL");
    if (!h->inited) return fail(h, RFLBM_ESTATE, "rflbm_get_populations before init");
    RFLBM_REQUIRE_HALO(h);
    return (h->precision == RFLBM_F64) ? do_export<double>(h, f_dev) : do_export<float>(h, f_dev);
}

// ---------------------------------------------------------------- the time step
// AUTO: the TMA kernel pays off when there is a long collision to hide the transfer behind; the deterministic
// kT = 0 update is pure streaming and the plain kernel's 20+ resident warps do better (8.72 vs 9.25 ms at 512^3)
static bool use_tma(const rflbm* h)
{
    if (!h->tma_ok || h->variant == RFLBM_KERNEL_PLAIN) return false;
    return h->variant == RFLBM_KERNEL_TMA || h->kT > 0.0;
}

// the step kernels are instantiated in rflbm_step_inst.cu, one translation unit per (precision, phase, tile width)
#define RFLBM_EXTERN_INST(R, PH)                                                                     \
    extern template void dispatch_variant<R, PH, 0>(rflbm*, const StepParams<R>&, int);              \
    extern template void dispatch_variant<R, PH, 32>(rflbm*, const StepParams<R>&, int);             \
    extern template void dispatch_variant<R, PH, 64>(rflbm*, const StepParams<R>&, int);             \
    extern template void dispatch_variant<R, PH, 128>(rflbm*, const StepParams<R>&, int);
RFLBM_EXTERN_INST(double, STEP_AB)
RFLBM_EXTERN_INST(double, STEP_AA_EVEN)
RFLBM_EXTERN_INST(double, STEP_AA_ODD)
RFLBM_EXTERN_INST(float, STEP_AB)
RFLBM_EXTERN_INST(float, STEP_AA_EVEN)
RFLBM_EXTERN_INST(float, STEP_AA_ODD)

template <typename real, int PHASE>
static void dispatch_tile(rflbm* h, const StepParams<real>& P, int variant, int tx)
{
    if (tx == 128) dispatch_variant<real, PHASE, 128>(h, P, variant);
    else if (tx == 64) dispatch_variant<real, PHASE, 64>(h, P, variant);
    else if (tx == 32) dispatch_variant<real, PHASE, 32>(h, P, variant);
    else dispatch_variant<real, PHASE, 0>(h, P, variant);
}

template <typename real>
static void dispatch_step(rflbm* h, const StepParams<real>& P, int variant, int tx)
{
    if (h->scheme == RFLBM_SCHEME_AB) dispatch_tile<real, STEP_AB>(h, P, variant, tx);
    else if (h->aa_phase == 0) dispatch_tile<real, STEP_AA_EVEN>(h, P, variant, tx);
    else dispatch_tile<real, STEP_AA_ODD>(h, P, variant, tx);
}

// one launch of the step kernel at time h->t over the owned layers [h->zc, h->zc + h->zn), reading buf[h->cur];
// no state change
template <typename real>
static int launch_step_once(rflbm* h)
{
    const bool noise = h->kT > 0.0;       // kT = 0: deterministic (Reg-)LBM, RNG skipped entirely (R17)
    if (h->variant == RFLBM_KERNEL_TMA && !h->tma_ok)
        return fail(h, RFLBM_EINVAL, "the TMA kernel needs nx >= 32 (and a driver that exports cuTensorMapEncodeTiled)");
    const bool tma = use_tma(h);
    const bool ghost = h->model == RFLBM_MODEL_REG && h->tau_g != 1.0;
    const int variant = (ghost ? 16 : 0) | (h->model == RFLBM_MODEL_BGK ? 8 : 0) | (h->walls ? 4 : 0) | (h->force ? 2 : 0) | (noise ? 1 : 0);
    static const char* const names[4] = {"step_kernel", "step_kernel_tma<TX=32>", "step_kernel_tma<TX=64>", "step_kernel_tma<TX=128>"};
    const StepParams<real> P = step_params<real>(h, h->t);
    dispatch_step<real>(h, P, variant, tma ? h->tma_tx : 0);
    h->last_kernel = !tma ? names[0] : h->tma_tx == 32 ? names[1] : h->tma_tx == 64 ? names[2] : names[3];
    return after_launch(h, h->last_kernel);
}

template <typename real>
static int do_step(rflbm* h, int nsteps)
{
    for (int s = 0; s < nsteps; ++s) {
        const int rc = launch_step_once<real>(h);
        if (rc != RFLBM_OK) return rc;
        if (h->scheme == RFLBM_SCHEME_AB) h->cur ^= 1;
        else h->aa_phase ^= 1;
        h->t += 1;
        if (h->slab) {
            h->halo_done = 0;
            h->halo_mode = (h->scheme == RFLBM_SCHEME_AB || h->aa_phase == 1) ? HALO_FILL : HALO_HOME;
        }
    }
    return RFLBM_OK;
}

extern "C" int rflbm_step(rflbm_t* h, int nsteps)
{
    if (!h) return RFLBM_EINVAL;
    if (nsteps < 0) return fail(h, RFLBM_EINVAL, "nsteps < 0");
    if (!h->inited) return fail(h, RFLBM_ESTATE, "rflbm_step before init");
    if (h->slab && nsteps > 1) return fail(h, RFLBM_EINVAL, "slab: one step at a time (the halos are exchanged between steps)");
    if (nsteps > 0) RFLBM_REQUIRE_HALO(h);
    return (h->precision == RFLBM_F64) ? do_step<double>(h, nsteps) : do_step<float>(h, nsteps);
}

// ---------------------------------------------------------------- observables
template <typename real>
static int do_moments(rflbm* h, void* rho, void* u)
{
    const FieldParams<real> P = field_params<real>(h);
    RFLBM_LAUNCH_OBSERVABLE(moments_kernel, (const real*)h->buf[h->cur], (real*)rho, (real*)u, P);
    return after_launch(h, "moments_kernel");
}

extern "C" int rflbm_moments(rflbm_t* h, void* rho_dev, void* u_dev)
{
    if (!h) return RFLBM_EINVAL;
    if (!rho_dev || !u_dev) return fail(h, RFLBM_EINVAL, "rho_dev / u_dev is NULL");
    if (!h->inited) return fail(h, RFLBM_ESTATE, "rflbm_moments before init");
    RFLBM_REQUIRE_HALO(h);
    return (h->precision == RFLBM_F64) ? do_moments<double>(h, rho_dev, u_dev) : do_moments<float>(h, rho_dev, u_dev);
}

template <typename real>
static int do_stress(rflbm* h, void* pi)
{
    const FieldParams<real> P = field_params<real>(h);
    RFLBM_LAUNCH_OBSERVABLE(stress_kernel, (const real*)h->buf[h->cur], (real*)pi, P);
    return after_launch(h, "stress_kernel");
}

extern "C" int rflbm_stress(rflbm_t* h, void* pi_dev)
{
    if (!h) return RFLBM_EINVAL;
    if (!pi_dev) return fail(h, RFLBM_EINVAL, "pi_dev is NULL");
    if (!h->inited) return fail(h, RFLBM_ESTATE, "rflbm_stress before init");
    RFLBM_REQUIRE_HALO(h);
    return (h->precision == RFLBM_F64) ? do_stress<double>(h, pi_dev) : do_stress<float>(h, pi_dev);
}

template <typename real>
static int do_snapshot(rflbm* h, void* rho, void* u, void* pi)
{
    const FieldParams<real> P = field_params<real>(h);
    RFLBM_LAUNCH_OBSERVABLE(snapshot_kernel, (const real*)h->buf[h->cur], (real*)rho, (real*)u, (real*)pi, P);
    return after_launch(h, "snapshot_kernel");
}

extern "C" int rflbm_snapshot(rflbm_t* h, void* rho_dev, void* u_dev, void* pi_dev)
{
    if (!h) return RFLBM_EINVAL;
    if (!rho_dev || !u_dev || !pi_dev) return fail(h, RFLBM_EINVAL, "rho_dev / u_dev / pi_dev is NULL");
    if (!h->inited) return fail(h, RFLBM_ESTATE, "rflbm_snapshot before init");
    RFLBM_REQUIRE_HALO(h);
    return (h->precision == RFLBM_F64) ? do_snapshot<double>(h, rho_dev, u_dev, pi_dev) : do_snapshot<float>(h, rho_dev, u_dev, pi_dev);
}

template <typename real>
static int do_diagnostics(rflbm* h)
{
    const FieldParams<real> P = field_params<real>(h);
    // every block walks the layers z = blockIdx.z, blockIdx.z + DIAG_ZBLOCKS, ... of its (x, y) patch
    const dim3 grid(h->grid.x, h->grid.y, (unsigned)std::min(h->zn, (int)DIAG_ZBLOCKS));
    RFLBM_LAUNCH_OBSERVABLE_GRID(grid, diagnostics_kernel, (const real*)h->buf[h->cur], h->acc, P, h->zn);
    return after_launch(h, "diagnostics_kernel");
}

extern "C" int rflbm_diagnostics(rflbm_t* h, double out_host[10])
{
    if (!h) return RFLBM_EINVAL;
    if (!out_host) return fail(h, RFLBM_EINVAL, "out_host is NULL");
    if (!h->inited) return fail(h, RFLBM_ESTATE, "rflbm_diagnostics before init");
    RFLBM_REQUIRE_HALO(h);
    static_assert(DIAG_ROWS * DIAG_PITCH * sizeof(double) == 4096, "the diagnostics rows fill the 4 KiB scratch");
    int rc = check_cuda(h, cudaMemsetAsync(h->acc, 0, 4096, h->stream), "cudaMemsetAsync");
    if (rc != RFLBM_OK) return rc;
    rc = (h->precision == RFLBM_F64) ? do_diagnostics<double>(h) : do_diagnostics<float>(h);
    if (rc != RFLBM_OK) return rc;
    double rows[DIAG_ROWS * DIAG_PITCH];
    rc = check_cuda(h, cudaMemcpyAsync(rows, h->acc, sizeof(rows), cudaMemcpyDeviceToHost, h->stream), "cudaMemcpyAsync");
    if (rc != RFLBM_OK) return rc;
    rc = check_cuda(h, cudaStreamSynchronize(h->stream), "cudaStreamSynchronize");
    if (rc != RFLBM_OK) return rc;
    double s[10];
    for (int n = 0; n < 10; ++n) {
        s[n] = 0.0;
        for (int r = 0; r < DIAG_ROWS; ++r) s[n] += rows[r * DIAG_PITCH + n];
    }
    // fluid layers owned by this handle (solid layers are global z = 0 and nz_global - 1)
    const int z0 = h->slab ? h->z0 : 0, nzg = h->slab ? h->nzg : h->nz;
    const int nfl = h->nz - (h->walls ? (z0 == 0) + (z0 + h->nz == nzg) : 0);
    const double nf = (double)h->nx * h->ny * nfl;
    out_host[0] = s[0];
    for (int a = 0; a < 3; ++a) {
        out_host[1 + a] = s[1 + a];
        // a slab that owns nothing but a solid layer has no fluid site: sums 0, mean and variance reported as 0
        out_host[4 + a] = nf > 0.0 ? s[4 + a] / nf : 0.0;
        out_host[7 + a] = nf > 0.0 ? s[7 + a] / nf - out_host[4 + a] * out_host[4 + a] : 0.0;
    }
    return RFLBM_OK;
}

extern "C" int rflbm_debug_rng(rflbm_t* h, uint64_t step, void* words_dev, void* normals_dev)
{
    if (!h) return RFLBM_EINVAL;
    if (!h->ws) return fail(h, RFLBM_ESTATE, "rflbm_debug_rng before rflbm_set_workspace");
    // acc[16] counts the sites where the hand-scheduled Philox differs from the textbook loop
    unsigned long long* mismatch = (unsigned long long*)(h->acc + 16);
    int rc = check_cuda(h, cudaMemsetAsync(mismatch, 0, sizeof(*mismatch), h->stream), "cudaMemsetAsync");
    if (rc != RFLBM_OK) return rc;
    const uint32_t t_hi = (uint32_t)(step >> 32), t_lo = (uint32_t)(step & 0xFFFFFFFFu);
    if (h->precision == RFLBM_F64) {
        const StepParams<double> P = step_params<double>(h, step);
        debug_rng_kernel<double><<<zgrid(h), h->block, 0, h->stream>>>((uint32_t*)words_dev, (double*)normals_dev,
                                                                     mismatch, t_hi, t_lo, P);
    } else {
        const StepParams<float> P = step_params<float>(h, step);
        debug_rng_kernel<float><<<zgrid(h), h->block, 0, h->stream>>>((uint32_t*)words_dev, (float*)normals_dev,
                                                                    mismatch, t_hi, t_lo, P);
    }
    rc = after_launch(h, "debug_rng_kernel");
    if (rc != RFLBM_OK) return rc;
    unsigned long long bad = 0;
    rc = check_cuda(h, cudaMemcpyAsync(&bad, mismatch, sizeof(bad), cudaMemcpyDeviceToHost, h->stream), "cudaMemcpyAsync");
    if (rc != RFLBM_OK) return rc;
    rc = check_cuda(h, cudaStreamSynchronize(h->stream), "cudaStreamSynchronize");
    if (rc != RFLBM_OK) return rc;
    if (bad != 0) return fail(h, RFLBM_ECUDA, "hand-scheduled Philox differs from the ten-round loop at %llu sites", bad);
    return RFLBM_OK;
}

// ---------------------------------------------------------------- host-buffer job (bench.py "e2e")
// Serial form: everything on the handle's stream, one copy after the other.
static int run_host_serial(rflbm* h, const void* rho_host, const void* u_host, int nsteps, void* rho_out_host,
                           void* u_out_host, char* d_rho, char* d_u, size_t fb)
{
    int rc;
    if (rho_host) {
        rc = check_cuda(h, cudaMemcpyAsync(d_rho, rho_host, fb, cudaMemcpyHostToDevice, h->stream), "H2D rho");
        if (rc != RFLBM_OK) return rc;
        rc = check_cuda(h, cudaMemcpyAsync(d_u, u_host, 3 * fb, cudaMemcpyHostToDevice, h->stream), "H2D u");
        if (rc != RFLBM_OK) return rc;
        rc = rflbm_init(h, d_rho, d_u);
    } else {
        rc = rflbm_init(h, nullptr, nullptr);
    }
    if (rc != RFLBM_OK) return rc;
    rc = rflbm_step(h, nsteps);
    if (rc != RFLBM_OK) return rc;
    rc = rflbm_moments(h, d_rho, d_u);
    if (rc != RFLBM_OK) return rc;
    rc = check_cuda(h, cudaMemcpyAsync(rho_out_host, d_rho, fb, cudaMemcpyDeviceToHost, h->stream), "D2H rho");
    if (rc != RFLBM_OK) return rc;
    rc = check_cuda(h, cudaMemcpyAsync(u_out_host, d_u, 3 * fb, cudaMemcpyDeviceToHost, h->stream), "D2H u");
    if (rc != RFLBM_OK) return rc;
    return check_cuda(h, cudaStreamSynchronize(h->stream), "cudaStreamSynchronize");
}

// Pipelined form (A-B scheme, a copy stream given): time-skewed along z.  The copies run on the copy stream, the kernels
// on the handle's stream, ordered by events.  Call "level L" the state after L steps (level 0: initialised; level L of
// layer z lives in buffer L & 1).  Bringing layers [a, b) to level L reads level L-1 on [a-1, b+1) — the pull reaches one
// layer up and down — and overwrites level L-2 there, which nobody needs once level L-1 is complete on [a-1, b+1).  So as
// soon as the layers [0, U) of (rho, u) are on the device, level L can be completed on [L+1, U-1-L): every band of CH
// uploaded layers lets EVERY level advance by CH layers, each one layer behind the level below it (a parallelogram in
// (z, t)), and the moments of the layers that have reached the last level go back to the host while the rest is still
// on the wire or stepping.  The ring is periodic, so one triangular seam stays open (level L is missing on
// [nz-1-L, nz) and [0, L+1)) until the last band has arrived; it is closed level by level at the end.  For long jobs
// only the first and the last SKEW levels are skewed (enough kernel time per band to hide the copies) and the levels
// in between run as whole-lattice launches.  Every launch is the same kernel restricted to a z range (Geom::zc), so the
// result is bit-identical to the serial form.
namespace {
template <typename real>
struct SkewJob {
    rflbm* h;
    const void *d_rho, *d_u;      // device fields for init (NULL: uniform start)
    int rc;
    // bring layers [a, b) from level L-1 to level L (L = 0: initialise from the uploaded fields)
    void level(int L, int a, int b)
    {
        if (rc != RFLBM_OK || b <= a) return;
        h->zc = a; h->zn = b - a;
        if (L == 0) {
            rc = do_init<real>(h, d_rho, d_u);
        } else {
            h->t = (uint64_t)(L - 1);
            h->cur = (L - 1) & 1;
            rc = launch_step_once<real>(h);
        }
    }
    // Levels base+1 .. base+n over the ring of nz layers, in bands of CH layers.  ready(U) is called before anything
    // that needs layers [0, U) of level `base` (the upload pass waits for the copy there; for a level that is complete
    // everywhere it does nothing); emit(a, b) is called once for every range of layers whose level base+n is final on
    // [a-1, b+1) (the moments can be taken).
    template <typename Ready, typename Emit>
    void pass(int base, int n, int CH, Ready ready, Emit emit)
    {
        const int nz = h->nz;
        int* hi = new (std::nothrow) int[n + 1];             // level base+i is done on [i, hi[i])
        if (!hi) { rc = RFLBM_ENOMEM; return; }
        for (int i = 0; i <= n; ++i) hi[i] = i;
        int out_hi = n + 1;                                  // emitted so far: [n+1, out_hi)
        for (int U = (CH < nz ? CH : nz);; U = (U + CH < nz ? U + CH : nz)) {
            ready(U);
            for (int i = 1; i <= n && i < U - i; ++i)
                if (U - i > hi[i]) { level(base + i, hi[i], U - i); hi[i] = U - i; }
            if (hi[n] - 1 > out_hi) { emit(out_hi, hi[n] - 1); out_hi = hi[n] - 1; }
            if (U == nz) break;
        }
        for (int i = 1; i <= n; ++i) {                       // the seam, level by level
            if (hi[i] <= i) level(base + i, 0, nz);
            else { level(base + i, hi[i], nz); level(base + i, 0, i); }
        }
        if (out_hi <= n + 1) emit(0, nz);
        else { emit(out_hi, nz); emit(0, n + 1); }
        delete[] hi;
    }
};
}  // namespace

template <typename real>
static int run_host_pipelined(rflbm* h, const void* rho_host, const void* u_host, int nsteps, void* rho_out_host,
                              void* u_out_host, char* d_rho, char* d_u, size_t fb)
{
    const size_t es = sizeof(real);
    // bands: at most 32, and thick enough that one band launch is ~8 waves of blocks (148 SMs x 3 blocks of the fp64 kernel;
    // 8 rows per block in a band launch), at least 4 bands where the lattice has the layers: 16 layers at 512^3 (measured
    // there, K = 20: 8 / 12 / 16 / 32 / 48 bands 240 / 239 / 237 / 238 / 243 ms), 56 at 256^3
    constexpr int MAXC = 32;
    // levels skewed at either end of a long job: a band of CH layers costs SKEW launches of ~1/32 step each, which has to
    // cover the copy of the band (2.4 ms of PCIe time against 0.3 ms per band and level at 512^3 fp64)
    constexpr int SKEW = 12;
    const int K = nsteps;
    const int tx = h->tma_tx ? h->tma_tx : 128;
    const long long blocks_per_layer = (long long)((h->nx + tx - 1) / tx) * ((h->ny + 7) / 8);
    int CH = (h->nz + MAXC - 1) / MAXC;
    const int thick = (int)std::min<long long>((8 * 444 + blocks_per_layer - 1) / blocks_per_layer, h->nz);
    if (thick > CH) CH = thick;
    if (CH > h->nz / 4) CH = h->nz / 4 > 0 ? h->nz / 4 : 1;
    const int C = (h->nz + CH - 1) / CH;
    const size_t layer = (size_t)h->nx * h->ny * es;
    // Every CUDA call below goes through ck(): the first failure is kept in job.rc (with its text in the handle), and
    // everything after it is skipped (SkewJob::level and the lambdas test job.rc).
    SkewJob<real> job{h, rho_host ? d_rho : nullptr, rho_host ? d_u : nullptr, RFLBM_OK};
    auto ck = [&](cudaError_t e, const char* what) {
        if (h->inject_fail > 0 && --h->inject_fail == 0 && e == cudaSuccess) e = cudaErrorUnknown;    // rflbm_debug_inject_failure
        if (e != cudaSuccess && job.rc == RFLBM_OK) job.rc = check_cuda(h, e, what);
        return e == cudaSuccess;
    };
    cudaEvent_t up[MAXC], start = nullptr, mom = nullptr;
    int n_up = 0;
    if (C > MAXC) job.rc = fail(h, RFLBM_EINVAL, "rflbm_run_host: %d bands", C);       // cannot happen: CH >= nz / 32
    while (job.rc == RFLBM_OK && n_up < C && ck(cudaEventCreateWithFlags(&up[n_up], cudaEventDisableTiming), "cudaEventCreate")) ++n_up;
    if (job.rc == RFLBM_OK && !ck(cudaEventCreateWithFlags(&start, cudaEventDisableTiming), "cudaEventCreate")) start = nullptr;
    if (job.rc == RFLBM_OK && !ck(cudaEventCreateWithFlags(&mom, cudaEventDisableTiming), "cudaEventCreate")) mom = nullptr;
    // a band launch is small: finer blocks (8 rows instead of 16) keep its last wave of blocks short
    const int rows_full = h->tma_rows;
    cudaStream_t cs = h->copy_stream;
    // the copy stream starts after whatever the caller has already enqueued on the handle's stream
    if (job.rc == RFLBM_OK) ck(cudaEventRecord(start, h->stream), "cudaEventRecord");
    if (job.rc == RFLBM_OK) ck(cudaStreamWaitEvent(cs, start, 0), "cudaStreamWaitEvent (copy stream)");
    // ---- uploads, in z order
    for (int c = 0; c < C && job.rc == RFLBM_OK; ++c) {
        if (rho_host) {
            const size_t off = (size_t)c * CH * layer, len = (size_t)((c == C - 1 ? h->nz - c * CH : CH)) * layer;
            ck(cudaMemcpyAsync(d_rho + off, (const char*)rho_host + off, len, cudaMemcpyHostToDevice, cs), "H2D rho");
            for (int k = 0; k < 3 && job.rc == RFLBM_OK; ++k)
                ck(cudaMemcpyAsync(d_u + k * fb + off, (const char*)u_host + k * fb + off, len, cudaMemcpyHostToDevice, cs), "H2D u");
        }
        if (job.rc == RFLBM_OK) ck(cudaEventRecord(up[c], cs), "cudaEventRecord (upload)");
    }
    auto uploaded = [&](int U) {
        if (job.rc == RFLBM_OK) ck(cudaStreamWaitEvent(h->stream, up[(U + CH - 1) / CH - 1], 0), "cudaStreamWaitEvent (upload)");
    };
    auto nothing = [](int) {};
    auto keep = [](int, int) {};
    // moments of layers [a, b) at the final level, then their way back to the host behind an event.  The downloads share
    // the copy stream with the uploads, which were all enqueued above: a download starts once the last band is up.
    auto output = [&](int a, int b) {
        if (job.rc != RFLBM_OK || b <= a) return;
        h->zc = a; h->zn = b - a;
        h->t = (uint64_t)K; h->cur = K & 1;
        job.rc = do_moments<real>(h, d_rho, d_u);
        if (job.rc != RFLBM_OK) return;
        if (!ck(cudaEventRecord(mom, h->stream), "cudaEventRecord (moments)")) return;
        if (!ck(cudaStreamWaitEvent(cs, mom, 0), "cudaStreamWaitEvent (moments)")) return;
        const size_t off = (size_t)a * layer, len = (size_t)(b - a) * layer;
        if (!ck(cudaMemcpyAsync((char*)rho_out_host + off, d_rho + off, len, cudaMemcpyDeviceToHost, cs), "D2H rho")) return;
        for (int k = 0; k < 3; ++k)
            if (!ck(cudaMemcpyAsync((char*)u_out_host + k * fb + off, d_u + k * fb + off, len, cudaMemcpyDeviceToHost, cs), "D2H u")) return;
    };
    if (job.rc == RFLBM_OK) {
        h->tma_rows = 8;
        if (K <= 2 * SKEW) {
            job.pass(-1, K + 1, CH, uploaded, output);              // one pass: init and all K steps behind the upload front
        } else {
            job.pass(-1, SKEW + 1, CH, uploaded, keep);             // init and the first SKEW steps behind the upload front
            h->tma_rows = rows_full;
            for (int L = SKEW + 1; L <= K - SKEW; ++L) job.level(L, 0, h->nz);      // whole-lattice launches
            h->tma_rows = 8;
            job.pass(K - SKEW, SKEW, CH, nothing, output);          // the last SKEW steps with the download behind them
        }
    }
    // ---- wait for both streams whatever happened (the caller's buffers must be quiet when the call returns)
    const cudaError_t e1 = cudaStreamSynchronize(cs), e2 = cudaStreamSynchronize(h->stream);
    for (int c = 0; c < n_up; ++c) cudaEventDestroy(up[c]);
    if (start) cudaEventDestroy(start);
    if (mom) cudaEventDestroy(mom);
    ck(e1, "cudaStreamSynchronize (copy stream)");
    ck(e2, "cudaStreamSynchronize");
    h->zc = 0; h->zn = h->nz;
    h->tma_rows = rows_full;
    h->inject_fail = 0;
    if (job.rc != RFLBM_OK) {
        // a job that failed half way leaves levels mixed over the layers: the handle holds no state (ESTATE until the
        // next rflbm_init / rflbm_set_populations / rflbm_run_host); the error text stays that of the first failure
        h->inited = false;
        h->t = 0; h->cur = 0; h->aa_phase = 0;
        cudaGetLastError();
        return job.rc;
    }
    // ---- state of the handle: as after rflbm_init + rflbm_step(nsteps)
    h->t = (uint64_t)nsteps; h->cur = nsteps & 1; h->aa_phase = 0; h->inited = true;
    after_state_change(h);
    return RFLBM_OK;
}

extern "C" int rflbm_run_host(rflbm_t* h, const void* rho_host, const void* u_host, int nsteps, void* rho_out_host,
                              void* u_out_host, void* scratch_dev, size_t scratch_bytes)
{
    if (!h) return RFLBM_EINVAL;
    if (!rho_out_host || !u_out_host || !scratch_dev) return fail(h, RFLBM_EINVAL, "NULL output or scratch pointer");
    if ((rho_host == nullptr) != (u_host == nullptr))
        return fail(h, RFLBM_EINVAL, "rho_host and u_host must both be given or both NULL");
    if (nsteps < 0) return fail(h, RFLBM_EINVAL, "nsteps < 0");
    if (!h->ws) return fail(h, RFLBM_ESTATE, "rflbm_run_host before rflbm_set_workspace");
    if (h->slab) return fail(h, RFLBM_ESTATE, "rflbm_run_host is a whole-lattice job: not available in slab mode");
    const size_t fb = (size_t)h->N * real_size(h);
    if (scratch_bytes < 4 * fb) return fail(h, RFLBM_ENOMEM, "scratch too small: %zu < %zu bytes", scratch_bytes, 4 * fb);
    char* d_rho = (char*)scratch_dev;
    char* d_u = d_rho + fb;
    // the pipeline needs a second stream, the A-B scheme (an odd AA step writes into its neighbours' layers) and at
    // least three chunks (a chunk's two neighbours must be two different chunks)
    if (h->copy_stream != nullptr && h->copy_stream != h->stream && h->scheme == RFLBM_SCHEME_AB && h->nz >= 3)
        return (h->precision == RFLBM_F64)
                   ? run_host_pipelined<double>(h, rho_host, u_host, nsteps, rho_out_host, u_out_host, d_rho, d_u, fb)
                   : run_host_pipelined<float>(h, rho_host, u_host, nsteps, rho_out_host, u_out_host, d_rho, d_u, fb);
    return run_host_serial(h, rho_host, u_host, nsteps, rho_out_host, u_out_host, d_rho, d_u, fb);
}

extern "C" int rflbm_debug_inject_failure(rflbm_t* h, int nth_call)
{
    if (!h) return RFLBM_EINVAL;
    if (nth_call < 0) return fail(h, RFLBM_EINVAL, "nth_call < 0");
    h->inject_fail = nth_call;
    return RFLBM_OK;
}

extern "C" int rflbm_set_copy_stream(rflbm_t* h, void* cuda_stream)
{
    if (!h) return RFLBM_EINVAL;
    h->copy_stream = (cudaStream_t)cuda_stream;
    return RFLBM_OK;
}

extern "C" int rflbm_set_scheme(rflbm_t* h, int scheme)
{
    if (!h) return RFLBM_EINVAL;
    if (scheme != RFLBM_SCHEME_AB && scheme != RFLBM_SCHEME_AA) return fail(h, RFLBM_EINVAL, "unknown scheme %d", scheme);
    if (h->ws) return fail(h, RFLBM_ESTATE, "rflbm_set_scheme must precede rflbm_set_workspace (the workspace size depends on it)");
    h->scheme = scheme;
    return RFLBM_OK;
}

// ---------------------------------------------------------------- z-slab decomposition
extern "C" int rflbm_set_slab(rflbm_t* h, int z0, int nz_global)
{
    if (!h) return RFLBM_EINVAL;
    if (h->ws) return fail(h, RFLBM_ESTATE, "rflbm_set_slab must precede rflbm_set_workspace (the workspace size depends on it)");
    if (z0 < 0 || nz_global < 1 || (long long)z0 + h->nz > nz_global)
        return fail(h, RFLBM_EINVAL, "slab [%d, %d) does not fit in %d global layers", z0, z0 + h->nz, nz_global);
    if ((double)h->nx * (double)h->ny * (double)nz_global >= 4294967296.0)
        return fail(h, RFLBM_EINVAL, "global lattice has 2^32 sites or more (the Philox site key is 32 bits, R8)");
    if (h->walls && nz_global < 3) return fail(h, RFLBM_EINVAL, "walls need nz_global >= 3");
    const int was = h->slab, was_z0 = h->z0, was_nzg = h->nzg;
    h->slab = 1; h->z0 = z0; h->nzg = nz_global;
    set_layout(h);
    if ((double)h->QS >= 4294967296.0) {
        h->slab = was; h->z0 = was_z0; h->nzg = was_nzg;
        set_layout(h);
        return fail(h, RFLBM_EINVAL, "slab too large");
    }
    return RFLBM_OK;
}

extern "C" size_t rflbm_halo_bytes(const rflbm_t* h)
{
    return h ? (size_t)9 * (size_t)h->nx * (size_t)h->ny * real_size(h) : 0;
}

extern "C" int rflbm_halo_pending(const rflbm_t* h) { return (h && halo_pending(h)) ? 1 : 0; }

// which storage layer and which 9 consecutive slots a face call touches (rflbm_kernels.cuh::halo_kernel).
// Storage layers: 0 = ghost below, 1..nz = owned, nz+1 = ghost above.  Slots 0..8 have c_z = -1, 18..26 c_z = +1.
//   HALO_FILL, A-B : the neighbour below pulls slot q (c_z = -1) of my bottom layer through its upper ghost
//   HALO_FILL, AA  : ... slot 26-q instead, i.e. the other nine
//   HALO_HOME (AA after an odd step): my lower ghost holds the c_z = -1 populations my bottom layer pushed down; they
//                    belong in slot q of the top layer of the neighbour below (and mirrored for the upper face)
// A buffer packed on one side is unpacked on the OTHER side of the neighbour with the same slots.
struct HaloPlan { int z, slot0; bool skip; };
static HaloPlan halo_plan(const rflbm* h, int side, bool pack)
{
    const bool ab = h->scheme == RFLBM_SCHEME_AB, low = side == RFLBM_SIDE_LOW;
    HaloPlan p;
    p.skip = false;
    if (h->halo_mode == HALO_FILL) {
        if (pack) { p.z = low ? 1 : h->nz; p.slot0 = (low == ab) ? 0 : 18; }
        else { p.z = low ? 0 : h->nz + 1; p.slot0 = (low == ab) ? 18 : 0; }
    } else {
        if (pack) { p.z = low ? 0 : h->nz + 1; p.slot0 = low ? 0 : 18; }
        else {
            p.z = low ? 1 : h->nz; p.slot0 = low ? 18 : 0;
            // nothing crosses a face next to a solid layer: a solid layer is never updated (it pushed nothing, and
            // keeps its values), and the fluid layer beside it bounced its populations back instead of pushing them
            const int zt = h->z0 + (low ? 0 : h->nz - 1);                                  // receiving layer
            const int zf = (zt + (low ? -1 : 1) + h->nzg) % h->nzg;                        // layer the data would come from
            p.skip = h->walls && (zt == 0 || zt == h->nzg - 1 || zf == 0 || zf == h->nzg - 1);
        }
    }
    return p;
}

template <bool PACK>
static int do_halo(rflbm* h, int side, void* face_dev)
{
    if (!h) return RFLBM_EINVAL;
    if (side != RFLBM_SIDE_LOW && side != RFLBM_SIDE_HIGH) return fail(h, RFLBM_EINVAL, "unknown side %d", side);
    if (!face_dev) return fail(h, RFLBM_EINVAL, "face_dev is NULL");
    if (!h->slab) return fail(h, RFLBM_ESTATE, "not in slab mode (rflbm_set_slab)");
    if (!h->inited) return fail(h, RFLBM_ESTATE, "halo call before init");
    if (h->halo_mode == HALO_NONE || (PACK && h->halo_done == 3)) return RFLBM_OK;    // nothing to exchange in this state
    // a side that has already been unpacked since the last step is complete: unpacking again would, in HALO_HOME,
    // overwrite nine populations of the boundary layer with whatever the face buffer holds by now
    if (!PACK && (h->halo_done & ((side == RFLBM_SIDE_LOW) ? 1 : 2))) return RFLBM_OK;
    const HaloPlan p = halo_plan(h, side, PACK);
    if (!p.skip) {
        const Geom G = make_geom(h);
        const dim3 grid(h->grid.x, h->grid.y, 1);
        if (h->precision == RFLBM_F64)
            halo_kernel<double, PACK><<<grid, h->block, 0, h->stream>>>((double*)h->buf[h->cur], (double*)face_dev, G, p.z, p.slot0);
        else
            halo_kernel<float, PACK><<<grid, h->block, 0, h->stream>>>((float*)h->buf[h->cur], (float*)face_dev, G, p.z, p.slot0);
        const int rc = after_launch(h, PACK ? "halo_kernel<pack>" : "halo_kernel<unpack>");
        if (rc != RFLBM_OK) return rc;
    }
    if (!PACK) h->halo_done |= (side == RFLBM_SIDE_LOW) ? 1 : 2;
    return RFLBM_OK;
}

extern "C" int rflbm_halo_pack(rflbm_t* h, int side, void* face_dev) { return do_halo<true>(h, side, face_dev); }
extern "C" int rflbm_halo_unpack(rflbm_t* h, int side, const void* face_dev) { return do_halo<false>(h, side, const_cast<void*>(face_dev)); }

extern "C" int rflbm_set_ghost_tau(rflbm_t* h, double tau_g)
{
    if (!h) return RFLBM_EINVAL;
    if (!std::isfinite(tau_g) || !(tau_g > 0.5)) return fail(h, RFLBM_EINVAL, "tau_g must be finite and > 0.5");
    if (tau_g != 1.0 && h->force) return fail(h, RFLBM_EINVAL, "the general ghost rate carries no body force");
    h->tau_g = tau_g;
    return RFLBM_OK;
}

extern "C" int rflbm_set_model(rflbm_t* h, int model)
{
    if (!h) return RFLBM_EINVAL;
    if (model != RFLBM_MODEL_REG && model != RFLBM_MODEL_BGK) return fail(h, RFLBM_EINVAL, "unknown model %d", model);
    if (model == RFLBM_MODEL_BGK && h->force) return fail(h, RFLBM_EINVAL, "BGK-FLBM carries no body force");
    h->model = model;
    return RFLBM_OK;
}

extern "C" int rflbm_set_kernel_variant(rflbm_t* h, int variant)
{
    if (!h) return RFLBM_EINVAL;
    if (variant != RFLBM_KERNEL_AUTO && variant != RFLBM_KERNEL_PLAIN && variant != RFLBM_KERNEL_TMA)
        return fail(h, RFLBM_EINVAL, "unknown kernel variant %d", variant);
    h->variant = variant;
    return RFLBM_OK;
}

// ---------------------------------------------------------------- misc
extern "C" uint64_t rflbm_launch_count(const rflbm_t* h) { return h ? h->launches : 0; }
extern "C" const char* rflbm_last_kernel(const rflbm_t* h) { return h ? h->last_kernel : ""; }
extern "C" uint64_t rflbm_step_count(const rflbm_t* h) { return h ? h->t : 0; }
extern "C" const char* rflbm_last_error(const rflbm_t* h) { return h ? h->err : "NULL handle"; }

extern "C" int rflbm_destroy(rflbm_t* h)
{
    if (!h) return RFLBM_EINVAL;
    delete h;
    return RFLBM_OK;
}
