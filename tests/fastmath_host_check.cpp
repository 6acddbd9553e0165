// fastmath_host_check.cpp — TEST SHIM: host build of csrc/rflbm_fastmath.cuh for tests/test_fastmath_host.py (CPU
// only; compiled by that test with -I paper_2507_08820_b200/csrc).
// Exposes the CUDA path's own Box-Muller pieces (compiled for the host) so that they can be compared with
// long-double libm over the whole 32-bit input range.  Not part of librflbm.so; shares nothing with oracle/.
#include "rflbm_fastmath.cuh"

using namespace rflbm_dev;

static f64x2 g_lg[LOG_TABLE_N], g_sc[SC_TABLE_N];
static bool g_ready = false;
static void ready()
{
    if (!g_ready) { fill_normal_tables(g_lg, g_sc); g_ready = true; }
}

extern "C" {
void fm_tables(double* lg, double* sc)
{
    ready();
    for (int j = 0; j < LOG_TABLE_N; ++j) { lg[2 * j] = g_lg[j].a; lg[2 * j + 1] = g_lg[j].b; }
    for (int j = 0; j < SC_TABLE_N; ++j) { sc[2 * j] = g_sc[j].a; sc[2 * j + 1] = g_sc[j].b; }
}
void fm_neg2_log(const uint32_t* x, double* out, long n)
{
    ready();
    for (long i = 0; i < n; ++i) out[i] = neg2_log_uniform(x[i], g_lg);
}
void fm_sqrt(const double* w, double* out, long n)
{
    for (long i = 0; i < n; ++i) out[i] = sqrt_pos(w[i]);
}
void fm_sincos(const uint32_t* x, double* s, double* c, long n)
{
    ready();
    for (long i = 0; i < n; ++i) sincos_uniform(x[i], g_sc, s[i], c[i]);
}
void fm_normal_pair(const uint32_t* xa, const uint32_t* xb, double* z0, double* z1, long n)
{
    ready();
    for (long i = 0; i < n; ++i) normal_pair_fast(xa[i], xb[i], g_lg, g_sc, z0[i], z1[i]);
}
}
