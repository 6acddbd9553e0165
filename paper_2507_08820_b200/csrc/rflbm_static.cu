// rflbm_static.cu — rflbm_diagnostics_static (include/rflbm.h): the conservation / velocity-variance sums of a
// canonical population field f[27][N], computed without a handle, without a workspace and without a single device
// allocation.
//
// Who this is for.  rflbm_diagnostics needs a handle, and a handle needs a workspace of one or two complete population
// buffers (29-58 GB at 512^3 fp64) that somebody has to allocate.  Some callers cannot: a restart tool or an in-situ
// monitor that is handed a checkpoint already sitting in device memory by a simulation that has claimed the rest of the
// HBM; a plug-in that runs inside a host application whose memory pool it may not touch; code on a path where
// cudaMalloc is forbidden because it synchronises the whole device (a latency-critical loop, a host callback).  For
// them the reduction scratch lives in THIS library's image: a file-scope __device__ array that the CUDA runtime
// places on every GPU that loads the library and that stays there until the process exits.
//
// The reduction is two launches on the caller's stream (no atomics, so the sums are the same bits every time):
//   stage 1  one block per 4096 sites: per-site moments (the same forward_moments as diagnostics_kernel), fp64 warp
//            shuffle + block sums -> s_static_scratch[block][10]
//   stage 2  one block: component n is summed over the blocks by warp n in a fixed order -> the last row of the array
// followed by an 80-byte copy to out_host and a stream synchronisation.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "../../include/rflbm.h"
#include "rflbm_collide.cuh"

using namespace rflbm_dev;

namespace {

constexpr int STATIC_THREADS = 256;
constexpr int STATIC_SITES_PER_THREAD = 16;
constexpr int STATIC_SITES_PER_BLOCK = STATIC_THREADS * STATIC_SITES_PER_THREAD;              // 4096
constexpr long long STATIC_MAX_SITES = RFLBM_STATIC_MAX_SITES;                                  // 2^27 = 512^3
constexpr int STATIC_MAX_BLOCKS = (int)(STATIC_MAX_SITES / STATIC_SITES_PER_BLOCK);           // 32 768
constexpr int STATIC_ROW = 10;                                                                  // doubles per block
constexpr int STATIC_MAX_DEVICES = 64;

// The scratch: one row of 10 partial sums per stage-1 block, plus one row for the result.  2 621 520 bytes (2.5 MiB)
// on every GPU that loads librflbm.so, for the life of the process.  Shared by every call on that GPU.
// NOTE for host code: `s_static_scratch` in a host function is the host-side shadow of the symbol, NOT a device
// address.  Host code must go through scratch_on_current_device() below; only device code may name the array.
static __device__ __align__(256) double s_static_scratch[(size_t)(STATIC_MAX_BLOCKS + 1) * STATIC_ROW];

// Device address of the array on each GPU, looked up once per device with that device current.
std::mutex s_mu;
double* s_scratch_addr[STATIC_MAX_DEVICES] = {};

int static_fail(char* err, size_t err_len, int code, const char* fmt, ...)
{
    if (err && err_len) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(err, err_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

// cudaGetSymbolAddress resolves the symbol for the CURRENT device; the result is cached per device ordinal.
cudaError_t scratch_on_current_device(double** out, int* dev_out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(s_mu);
    if (!s_scratch_addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, s_static_scratch);
        if (e != cudaSuccess) return e;
        s_scratch_addr[dev] = (double*)p;
    }
    *out = s_scratch_addr[dev];
    *dev_out = dev;
    return cudaSuccess;
}

struct StaticParams {
    long long N;        // sites
    long long nxy;      // nx*ny: z = s / nxy
    int nz;
    int walls;          // layers z = 0 and z = nz-1 are solid and left out (R12)
    double hg[3];       // g/2 (R13)
};

// stage 1: sums over the fluid sites of one 4096-site chunk of { rho, rho u_x,y,z, u_x,y,z, u_x^2,y^2,z^2 }
template <typename real>
__global__ void __launch_bounds__(STATIC_THREADS)
static_partial_kernel(const real* __restrict__ f, double* __restrict__ partial, const StaticParams P)
{
    double v[STATIC_ROW];
#pragma unroll
    for (int n = 0; n < STATIC_ROW; ++n) v[n] = 0.0;
    const long long base = (long long)blockIdx.x * STATIC_SITES_PER_BLOCK + threadIdx.x;
    for (int k = 0; k < STATIC_SITES_PER_THREAD; ++k) {
        const long long s = base + (long long)k * STATIC_THREADS;
        if (s >= P.N) break;
        if (P.walls) {
            const long long z = s / P.nxy;
            if (z == 0 || z == P.nz - 1) continue;
        }
        real g[3][3][3];
#pragma unroll
        for (int i = 0; i < Q; ++i) g[canon_cz(i) + 1][canon_cy(i) + 1][canon_cx(i) + 1] = __ldg(f + (long long)i * P.N + s);
        const Moments10<real> m = forward_moments(g);
        const double rho = (double)m.rho, inv = 1.0 / rho;     // one fp64 division per site, not three
        const double ux = fma((double)m.jx, inv, P.hg[0]);
        const double uy = fma((double)m.jy, inv, P.hg[1]);
        const double uz = fma((double)m.jz, inv, P.hg[2]);
        v[0] += rho; v[1] += rho * ux; v[2] += rho * uy; v[3] += rho * uz;
        v[4] += ux; v[5] += uy; v[6] += uz; v[7] += ux * ux; v[8] += uy * uy; v[9] += uz * uz;
    }
    __shared__ double part[STATIC_THREADS / 32][STATIC_ROW];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int n = 0; n < STATIC_ROW; ++n) {
        double s = v[n];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (lane == 0) part[warp][n] = s;
    }
    __syncthreads();
    if (threadIdx.x < STATIC_ROW) {
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < STATIC_THREADS / 32; ++w) s += part[w][threadIdx.x];
        partial[(size_t)blockIdx.x * STATIC_ROW + threadIdx.x] = s;          // every row a later read uses is written here first
    }
}

// stage 2: one block of 10 warps; warp n adds component n of the first `nblocks` rows in a fixed order
__global__ void __launch_bounds__(32 * STATIC_ROW)
static_final_kernel(const double* __restrict__ partial, double* __restrict__ result, int nblocks)
{
    const int lane = threadIdx.x & 31, n = threadIdx.x >> 5;
    double s = 0.0;
    for (int b = lane; b < nblocks; b += 32) s += partial[(size_t)b * STATIC_ROW + n];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) result[n] = s;
}

}  // namespace

extern "C" long long rflbm_static_max_sites(void) { return STATIC_MAX_SITES; }

extern "C" int rflbm_diagnostics_static(const void* f_dev, int nx, int ny, int nz, int precision, int walls_z,
                                        const double* g_host, void* cuda_stream, double out_host[10], char* err_host,
                                        size_t err_len)
{
    if (err_host && err_len) err_host[0] = '\0';
    // ---- host-only validation: nothing below this block runs for a rejected call
    if (!f_dev || !out_host) return static_fail(err_host, err_len, RFLBM_EINVAL, "f_dev / out_host is NULL");
    if (nx < 1 || ny < 1 || nz < 1) return static_fail(err_host, err_len, RFLBM_EINVAL, "nx, ny, nz must be >= 1");
    if (precision != RFLBM_F64 && precision != RFLBM_F32)
        return static_fail(err_host, err_len, RFLBM_EINVAL, "unknown precision %d", precision);
    const double sites = (double)nx * (double)ny * (double)nz;
    if (sites > (double)STATIC_MAX_SITES)
        return static_fail(err_host, err_len, RFLBM_EINVAL,
                           "lattice of %.0f sites exceeds the static scratch of rflbm_diagnostics_static: at most %lld sites "
                           "(512^3); use rflbm_diagnostics on a handle with a caller-allocated workspace instead",
                           sites, STATIC_MAX_SITES);
    if (walls_z && nz < 3) return static_fail(err_host, err_len, RFLBM_EINVAL, "walls need nz >= 3");
    StaticParams P;
    P.N = (long long)nx * ny * nz;
    P.nxy = (long long)nx * ny;
    P.nz = nz;
    P.walls = walls_z ? 1 : 0;
    for (int a = 0; a < 3; ++a) {
        const double g = g_host ? g_host[a] : 0.0;
        if (!std::isfinite(g)) return static_fail(err_host, err_len, RFLBM_EINVAL, "non-finite acceleration");
        // g/2 in `real`, as the handle's observables carry it (FieldParams::hgx): the two paths then add the same number
        P.hg[a] = (precision == RFLBM_F32) ? (double)(float)(0.5 * g) : 0.5 * g;
    }
    // ---- set-up (first call on this device): device address of the static array
    double* scratch = nullptr;
    int dev = -1;
    cudaError_t e = scratch_on_current_device(&scratch, &dev);
    if (e != cudaSuccess)
        return static_fail(err_host, err_len, RFLBM_ECUDA, "cudaGetSymbolAddress(static scratch): %s", cudaGetErrorString(e));
    cudaPointerAttributes attr;
    e = cudaPointerGetAttributes(&attr, f_dev);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return static_fail(err_host, err_len, RFLBM_EINVAL, "f_dev is not a CUDA pointer: %s", cudaGetErrorString(e));
    }
    if (attr.type != cudaMemoryTypeDevice && attr.type != cudaMemoryTypeManaged)
        return static_fail(err_host, err_len, RFLBM_EINVAL, "f_dev must be device memory");
    if (attr.type == cudaMemoryTypeDevice && attr.device != dev)
        return static_fail(err_host, err_len, RFLBM_EINVAL,
                           "f_dev lives on device %d but device %d is current: the static scratch is per device, make the "
                           "field's device current before the call", attr.device, dev);
    // ---- two launches + the read-back on the caller's stream
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    const int nblocks = (int)((P.N + STATIC_SITES_PER_BLOCK - 1) / STATIC_SITES_PER_BLOCK);      // <= STATIC_MAX_BLOCKS
    double* result = scratch + (size_t)STATIC_MAX_BLOCKS * STATIC_ROW;
    if (precision == RFLBM_F64)
        static_partial_kernel<double><<<nblocks, STATIC_THREADS, 0, stream>>>((const double*)f_dev, scratch, P);
    else
        static_partial_kernel<float><<<nblocks, STATIC_THREADS, 0, stream>>>((const float*)f_dev, scratch, P);
    static_final_kernel<<<1, 32 * STATIC_ROW, 0, stream>>>(scratch, result, nblocks);
    e = cudaPeekAtLastError();
    if (e != cudaSuccess) return static_fail(err_host, err_len, RFLBM_ECUDA, "launch: %s", cudaGetErrorString(e));
    double s[STATIC_ROW];
    e = cudaMemcpyAsync(s, result, sizeof(s), cudaMemcpyDeviceToHost, stream);
    if (e != cudaSuccess) return static_fail(err_host, err_len, RFLBM_ECUDA, "cudaMemcpyAsync: %s", cudaGetErrorString(e));
    e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) return static_fail(err_host, err_len, RFLBM_ECUDA, "cudaStreamSynchronize: %s", cudaGetErrorString(e));
    const double nf = (double)nx * ny * (nz - (walls_z ? 2 : 0));
    out_host[0] = s[0];
    for (int a = 0; a < 3; ++a) {
        out_host[1 + a] = s[1 + a];
        out_host[4 + a] = s[4 + a] / nf;
        out_host[7 + a] = s[7 + a] / nf - out_host[4 + a] * out_host[4 + a];
    }
    return RFLBM_OK;
}
