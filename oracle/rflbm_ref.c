/*
 * rflbm_ref.c — CPU ORACLE for the D3Q27 regularized fluctuating lattice Boltzmann
 * collide-and-stream step of arXiv 2507.08820.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or constant generator with the CUDA path under
 * paper_2507_08820_b200/csrc/.  It is deliberately plain and slow: dense 27x27
 * transforms, explicit loops, double everywhere, libm transcendentals, summation in
 * index order, no FMA contraction (build with -ffp-contract=off).
 *
 * What it follows (PAPER.md line : equation / table):
 *   lattice + weights            :70-77   Table I        (velocity order inside groups: DESIGN.md R1)
 *   Hermite basis e_ki, b_k      :172-202 Table II, :68 Eq.5   (rows 23,24,26: DESIGN.md R2)
 *   rho, rho u                   :56-58   Eq.2-3
 *   a_1,ab (2nd order neq)       :153     Eq.19  with Eq.18,20 (:150, :160)
 *   a_0^(n) = rho u..u           :160     Eq.20
 *   noise phi_k r_k, k=4..26     :93-99   Eq.8-9 (k=1..3 carry no noise, :95; R3)
 *   back-transform               :105     Eq.10 (== Eq.25+26, :225-229)
 *   final update                 :221     Eq.24  with omega_g = 1 (:215)
 *   general ghost rate omega_g   :163-166 Eq.21 recursion (perm: DESIGN.md R20), :211-215
 *   BGK-FLBM (comparison model)  :109-111 Eq.11 with Eq.6 (:85), in population space (f^eq: DESIGN.md R19)
 *   streaming                    :87      Eq.7   (periodic; bounce-back walls: DESIGN.md R12)
 *   body force (Guo, moment form): not in the paper, R13
 *   random numbers               : "standard normal" :95; generator + mapping: DESIGN.md R8
 *
 * Pins (tests/test_oracle_*.py, all run without a GPU): table identities in exact rational
 * arithmetic against the values printed in Table I/II; Philox4x32-10 known-answer vectors;
 * Box-Muller closed-form points and sample statistics; mass/momentum conservation;
 * equilibrium fixed point and product closed form; post-collision moment structure;
 * brute-force streaming on tiny boxes; Taylor-Green decay rate nu=(tau-1/2)/3;
 * equipartition of all 27 modes; flat structure factor; Poiseuille profile with walls+force;
 * diagnostics mean/variance over fluid sites against the printed basis rows 0..3 and closed forms
 * (tests/test_oracle_diagnostics.py); the fp32 storage mode: every stored value is a float after init
 * and after every step in all three store sites, one step = rounded single-site collision streamed by
 * numpy, 24-bit uniforms (tests/test_oracle_fp32.py).
 * Parity unpinned: near-wall fluctuation variance with walls (nothing fixes it).
 */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define Q 27
#define REF_OK 0
#define REF_EINVAL (-1)
#define REF_ESTATE (-2)
#define REF_ENOMEM (-3)

#define REF_F64 0
#define REF_F32 1

#define REF_MODEL_REG 0   /* Reg-FLBM, Eq.24: the hot path                         */
#define REF_MODEL_BGK 1   /* BGK-FLBM, Eq.11: the paper's comparison model      */

/* ------------------------------------------------------------------ tables */

static int    T_ready = 0;
static int    T_c[Q][3];      /* velocities, canonical order R1                  */
static double T_w[Q];         /* weights, Table I                                  */
static int    T_opp[Q];       /* c[opp[i]] = -c[i]                                 */
static int    T_pqr[Q][3];    /* Hermite exponents per mode, Table II order        */
static double T_e[Q][Q];      /* e[k][i] = H_p(c_ix) H_q(c_iy) H_r(c_iz)           */
static double T_b[Q];         /* b_k = sum_i w_i e_ki^2  (Eq.5)                    */

static double hermite1d(int p, int c)
{
    /* H_0 = 1, H_1 = c, H_2 = c^2 - c_s^2 with c_s^2 = 1/3 (Table II polynomials factorise
     * into these, R2) */
    if (p == 0) return 1.0;
    if (p == 1) return (double)c;
    return (double)(c * c) - 1.0 / 3.0;
}

static void build_tables(void)
{
    if (T_ready) return;
    int n = 0;
    const int sgn[2] = {+1, -1};
    /* 0: rest */
    T_c[n][0] = 0; T_c[n][1] = 0; T_c[n][2] = 0; n++;
    /* 1..6: +x,-x,+y,-y,+z,-z */
    for (int a = 0; a < 3; a++)
        for (int s = 0; s < 2; s++) {
            T_c[n][0] = T_c[n][1] = T_c[n][2] = 0;
            T_c[n][a] = sgn[s];
            n++;
        }
    /* 7..10 (sx,sy,0); 11..14 (sx,0,sz); 15..18 (0,sy,sz); sign order (+,+),(+,-),(-,+),(-,-) */
    const int pairs[3][2] = {{0, 1}, {0, 2}, {1, 2}};
    for (int pr = 0; pr < 3; pr++)
        for (int s1 = 0; s1 < 2; s1++)
            for (int s2 = 0; s2 < 2; s2++) {
                T_c[n][0] = T_c[n][1] = T_c[n][2] = 0;
                T_c[n][pairs[pr][0]] = sgn[s1];
                T_c[n][pairs[pr][1]] = sgn[s2];
                n++;
            }
    /* 19..26 (sx,sy,sz), sx outermost */
    for (int s1 = 0; s1 < 2; s1++)
        for (int s2 = 0; s2 < 2; s2++)
            for (int s3 = 0; s3 < 2; s3++) {
                T_c[n][0] = sgn[s1]; T_c[n][1] = sgn[s2]; T_c[n][2] = sgn[s3];
                n++;
            }
    for (int i = 0; i < Q; i++) {
        int c2 = T_c[i][0] * T_c[i][0] + T_c[i][1] * T_c[i][1] + T_c[i][2] * T_c[i][2];
        T_w[i] = (c2 == 0) ? 8.0 / 27.0 : (c2 == 1) ? 2.0 / 27.0 : (c2 == 2) ? 1.0 / 54.0 : 1.0 / 216.0;
        for (int j = 0; j < Q; j++)
            if (T_c[j][0] == -T_c[i][0] && T_c[j][1] == -T_c[i][1] && T_c[j][2] == -T_c[i][2]) T_opp[i] = j;
    }
    /* Table II order of (p,q,r) */
    static const int pqr[Q][3] = {
        {0,0,0},
        {1,0,0},{0,1,0},{0,0,1},
        {2,0,0},{0,2,0},{0,0,2},
        {1,1,0},{1,0,1},{0,1,1},
        {2,1,0},{2,0,1},{1,2,0},{1,0,2},{0,1,2},{0,2,1},
        {1,1,1},
        {2,2,0},{2,0,2},{0,2,2},
        {1,1,2},{1,2,1},{2,1,1},
        {2,1,2},{2,2,1},{1,2,2},
        {2,2,2}};
    for (int k = 0; k < Q; k++) {
        for (int a = 0; a < 3; a++) T_pqr[k][a] = pqr[k][a];
        double bk = 0.0;
        for (int i = 0; i < Q; i++) {
            T_e[k][i] = hermite1d(pqr[k][0], T_c[i][0]) * hermite1d(pqr[k][1], T_c[i][1]) *
                        hermite1d(pqr[k][2], T_c[i][2]);
            bk += T_w[i] * T_e[k][i] * T_e[k][i];
        }
        T_b[k] = bk;
    }
    T_ready = 1;
}

/* copies the tables out for the pin tests */
int rflbm_ref_tables(int *c /*[27][3]*/, double *w /*[27]*/, int *opp /*[27]*/, int *pqr /*[27][3]*/,
                     double *e /*[27][27]*/, double *b /*[27]*/)
{
    build_tables();
    for (int i = 0; i < Q; i++) {
        if (c) for (int a = 0; a < 3; a++) c[3 * i + a] = T_c[i][a];
        if (w) w[i] = T_w[i];
        if (opp) opp[i] = T_opp[i];
        if (pqr) for (int a = 0; a < 3; a++) pqr[3 * i + a] = T_pqr[i][a];
        if (b) b[i] = T_b[i];
        if (e) for (int j = 0; j < Q; j++) e[Q * i + j] = T_e[i][j];
    }
    return REF_OK;
}

/* ------------------------------------------------------------------ random numbers (R8) */

/* Philox4x32-10 as published (Salmon, Moraes, Dror, Shaw, SC'11). */
void rflbm_ref_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; round++) {
        if (round > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Box-Muller on two 32-bit words (R8).  fp64 mode: 32-bit uniforms (x+0.5)/2^32;
 * fp32 mode: 24-bit uniforms ((x>>8)+0.5)/2^24.  Arithmetic is double in both. */
void rflbm_ref_normal_pair(uint32_t xa, uint32_t xb, int precision, double out[2])
{
    double ua, ub;
    if (precision == REF_F32) {
        ua = ((double)(xa >> 8) + 0.5) * (1.0 / 16777216.0);
        ub = ((double)(xb >> 8) + 0.5) * (1.0 / 16777216.0);
    } else {
        ua = ((double)xa + 0.5) * (1.0 / 4294967296.0);
        ub = ((double)xb + 0.5) * (1.0 / 4294967296.0);
    }
    const double two_pi = 6.283185307179586476925286766559;
    double R = sqrt(-2.0 * log(ua));
    out[0] = R * cos(two_pi * ub);
    out[1] = R * sin(two_pi * ub);
}

/* the 24 words and 23 normals (modes 4..26) of one (site, step) */
static void draw_site(uint64_t seed, uint64_t t, uint32_t site, int precision, uint32_t words[24], double r[Q])
{
    uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32)};
    for (int k = 0; k < Q; k++) r[k] = 0.0;
    for (uint32_t q = 0; q < 6; q++) {
        uint32_t ctr[4] = {site, (uint32_t)(t >> 32), (uint32_t)(t & 0xFFFFFFFFu), q};
        uint32_t x[4];
        rflbm_ref_philox4x32_10(ctr, key, x);
        for (int m = 0; m < 4; m++) words[4 * q + m] = x[m];
        for (int h = 0; h < 2; h++) {
            double z[2];
            rflbm_ref_normal_pair(x[2 * h], x[2 * h + 1], precision, z);
            int k = 4 + 4 * (int)q + 2 * h;
            if (k < Q) r[k] = z[0];
            if (k + 1 < Q) r[k + 1] = z[1];   /* q=5,h=1: second value (k=27) is discarded */
        }
    }
}

/* ------------------------------------------------------------------ handle */

typedef struct rflbm_ref {
    int nx, ny, nz;
    double tau, kT, rho0;
    uint64_t seed;
    int precision;
    int walls_z;
    int model;    /* REF_MODEL_REG (Eq.24) or REF_MODEL_BGK (Eq.11) */
    double tau_g; /* ghost relaxation time 1/omega_g of Reg-FLBM; 0 or 1 = the paper's choice omega_g = 1 (:215) */
    double g[3];
    uint64_t t;
    int inited;
    double *S;    /* pre-collision populations f_i(x,t), canonical [27][nz][ny][nx] */
    double *S2;
    int nthreads;
    char err[256];
} rflbm_ref_t;

static size_t nsites(const rflbm_ref_t *h) { return (size_t)h->nx * h->ny * h->nz; }

static int is_solid(const rflbm_ref_t *h, int z) { return h->walls_z && (z == 0 || z == h->nz - 1); }

int rflbm_ref_create(int nx, int ny, int nz, double tau, double kT, double rho0, uint64_t seed, int precision,
                     rflbm_ref_t **out)
{
    if (!out) return REF_EINVAL;
    *out = NULL;
    if (nx < 1 || ny < 1 || nz < 1) return REF_EINVAL;
    if (!isfinite(tau) || !(tau > 0.5)) return REF_EINVAL;
    if (!isfinite(kT) || kT < 0.0) return REF_EINVAL;
    if (!isfinite(rho0) || !(rho0 > 0.0)) return REF_EINVAL;
    if (precision != REF_F64 && precision != REF_F32) return REF_EINVAL;
    if ((double)nx * ny * nz >= 4294967296.0) return REF_EINVAL;
    build_tables();
    rflbm_ref_t *h = (rflbm_ref_t *)calloc(1, sizeof(*h));
    if (!h) return REF_ENOMEM;
    h->nx = nx; h->ny = ny; h->nz = nz;
    h->tau = tau; h->kT = kT; h->rho0 = rho0; h->seed = seed; h->precision = precision;
    h->nthreads = 1;
    h->tau_g = 1.0;
    size_t n = nsites(h);
    h->S = (double *)malloc(sizeof(double) * Q * n);
    h->S2 = (double *)malloc(sizeof(double) * Q * n);
    if (!h->S || !h->S2) { free(h->S); free(h->S2); free(h); return REF_ENOMEM; }
    *out = h;
    return REF_OK;
}

int rflbm_ref_destroy(rflbm_ref_t *h)
{
    if (!h) return REF_EINVAL;
    free(h->S); free(h->S2); free(h);
    return REF_OK;
}

int rflbm_ref_set_threads(rflbm_ref_t *h, int n)
{
    if (!h || n < 1) return REF_EINVAL;
    h->nthreads = n;
    return REF_OK;
}

int rflbm_ref_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_num_procs();
#else
    return 1;
#endif
}

int rflbm_ref_set_walls_z(rflbm_ref_t *h, int on)
{
    if (!h) return REF_EINVAL;
    if (on && h->nz < 3) return REF_EINVAL;
    h->walls_z = on ? 1 : 0;
    return REF_OK;
}

int rflbm_ref_set_force(rflbm_ref_t *h, double gx, double gy, double gz)
{
    if (!h || !isfinite(gx) || !isfinite(gy) || !isfinite(gz)) return REF_EINVAL;
    if (h->model == REF_MODEL_BGK && (gx != 0.0 || gy != 0.0 || gz != 0.0)) return REF_EINVAL;
    h->g[0] = gx; h->g[1] = gy; h->g[2] = gz;
    return REF_OK;
}

int rflbm_ref_set_ghost_tau(rflbm_ref_t *h, double tau_g)
{
    if (!h || !isfinite(tau_g) || !(tau_g > 0.5)) return REF_EINVAL;
    h->tau_g = tau_g;
    return REF_OK;
}

int rflbm_ref_set_model(rflbm_ref_t *h, int model)
{
    if (!h || (model != REF_MODEL_REG && model != REF_MODEL_BGK)) return REF_EINVAL;
    if (model == REF_MODEL_BGK && (h->g[0] != 0.0 || h->g[1] != 0.0 || h->g[2] != 0.0)) return REF_EINVAL;
    h->model = model;
    return REF_OK;
}

uint64_t rflbm_ref_step_count(const rflbm_ref_t *h) { return h ? h->t : 0; }

static double store_round(const rflbm_ref_t *h, double v)
{
    /* fp32 storage mode (R14): the state is rounded to float whenever it is stored */
    return (h->precision == REF_F32) ? (double)(float)v : v;
}

/* Eq.25 :225 with Eq.20 :160 — f0_i = w_i sum_k rho ux^p uy^q uz^r e_ki / b_k */
void rflbm_ref_equilibrium(double rho, const double u[3], double f0[Q])
{
    build_tables();
    double M[Q];
    for (int k = 0; k < Q; k++) {
        double m = rho;
        for (int a = 0; a < 3; a++)
            for (int n = 0; n < T_pqr[k][a]; n++) m = m * u[a];
        M[k] = m;
    }
    for (int i = 0; i < Q; i++) {
        double s = 0.0;
        for (int k = 0; k < Q; k++) s += M[k] * T_e[k][i] / T_b[k];
        f0[i] = T_w[i] * s;
    }
}

int rflbm_ref_init(rflbm_ref_t *h, const double *rho, const double *u)
{
    if (!h) return REF_EINVAL;
    if ((rho == NULL) != (u == NULL)) return REF_EINVAL;
    size_t n = nsites(h);
    for (size_t s = 0; s < n; s++) {
        double r = rho ? rho[s] : h->rho0;
        double uu[3] = {0.0, 0.0, 0.0};
        if (u) { uu[0] = u[s]; uu[1] = u[n + s]; uu[2] = u[2 * n + s]; }
        double f0[Q];
        rflbm_ref_equilibrium(r, uu, f0);
        for (int i = 0; i < Q; i++) h->S[(size_t)i * n + s] = store_round(h, f0[i]);
    }
    h->t = 0;
    h->inited = 1;
    return REF_OK;
}

/* ------------------------------------------------------------------ collision at one site */

/* Eq.21, the recursive non-equilibrium Hermite coefficients of order n >= 3, literally:
 *   a1^(n)[a1..an] = a1^(n-1)[a1..a(n-1)] u[an] + ( u[a1]..u[a(n-2)] a1^(2)[a(n-1) an] + perm(an) ),
 * "perm(an)" = the permutations that pair an with each of the first n-1 indices in turn (reading R20: these are
 * the n-1 terms sum_j a1^(2)[aj an] prod_{k<n, k!=j} u[ak]; Malaspinas' recursive regularization, ref. 55).
 * Tensors of rank n are stored with 3^n entries, index = a1 3^(n-1) + ... + an.  A[2] is the input a1^(2). */
static void a1_recursion(const double a2[3][3], const double u[3], double A3[27], double A4[81], double A5[243],
                         double A6[729])
{
    double A2[9];
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) A2[3 * i + j] = a2[i][j];
    double *A[7] = {0, 0, A2, A3, A4, A5, A6};
    int size = 9;
    for (int n = 3; n <= 6; n++) {
        size *= 3;
        for (int idx = 0; idx < size; idx++) {
            int al[6], t = idx;
            for (int k = n - 1; k >= 0; k--) { al[k] = t % 3; t /= 3; }       /* al[0..n-1] = a1..an */
            double val = A[n - 1][idx / 3] * u[al[n - 1]];
            for (int j = 0; j < n - 1; j++) {
                double term = a2[al[j]][al[n - 1]];
                for (int k = 0; k < n - 1; k++)
                    if (k != j) term *= u[al[k]];
                val += term;
            }
            A[n][idx] = val;
        }
    }
}

/* coefficient of mode k = (p,q,r): the tensor entry with p x-indices, q y-indices, r z-indices (any order) */
static double a1_of_mode(int k, const double a2[3][3], const double A3[27], const double A4[81], const double A5[243],
                         const double A6[729])
{
    int al[6], n = 0;
    for (int a = 0; a < 3; a++)
        for (int m = 0; m < T_pqr[k][a]; m++) al[n++] = a;
    int idx = 0;
    for (int m = 0; m < n; m++) idx = 3 * idx + al[m];
    if (n == 2) return a2[al[0]][al[1]];
    return (n == 3) ? A3[idx] : (n == 4) ? A4[idx] : (n == 5) ? A5[idx] : A6[idx];
}

/* steps 2-7 of DESIGN.md "one step"; g = pre-collision populations of the site */
static void collide(const rflbm_ref_t *h, const double g[Q], uint32_t site, uint64_t t, double fstar[Q])
{
    const double omega_h = 1.0 / h->tau;
    const double cs2 = 1.0 / 3.0;

    /* 2. conserved moments, Eq.2-3 */
    double rho = 0.0, j[3] = {0.0, 0.0, 0.0};
    for (int i = 0; i < Q; i++) rho += g[i];
    for (int a = 0; a < 3; a++)
        for (int i = 0; i < Q; i++) j[a] += g[i] * (double)T_c[i][a];
    double F[3], u[3];
    for (int a = 0; a < 3; a++) {
        F[a] = rho * h->g[a];
        u[a] = (j[a] + 0.5 * F[a]) / rho;
    }

    /* 3. second-order non-equilibrium Hermite coefficients, Eq.19 with Eq.18, 20 */
    static const int AB[6][2] = {{0, 0}, {1, 1}, {2, 2}, {0, 1}, {0, 2}, {1, 2}}; /* k=4..9 */
    double a1[6];
    for (int m = 0; m < 6; m++) {
        int a = AB[m][0], b = AB[m][1];
        double s = 0.0;
        for (int i = 0; i < Q; i++)
            s += g[i] * ((double)(T_c[i][a] * T_c[i][b]) - (a == b ? cs2 : 0.0));
        a1[m] = s - rho * u[a] * u[b];
    }

    /* 4. equilibrium Hermite coefficients, Eq.20 */
    double M[Q];
    for (int k = 0; k < Q; k++) {
        double m = rho;
        for (int a = 0; a < 3; a++)
            for (int n = 0; n < T_pqr[k][a]; n++) m = m * u[a];
        M[k] = m;
    }

    /* 5. relaxed hydrodynamic non-equilibrium part, Eq.26 with (1-omega_h), Eq.24; ghosts: 1-omega_g = 0 */
    for (int m = 0; m < 6; m++) M[4 + m] += (1.0 - omega_h) * a1[m];
    /* general ghost rate (:211-215 before omega_g is set to 1): (1-omega_g) f^(1,g), the ghost part of Eq.17 with
     * the coefficients of Eq.21 */
    const double omega_g = (h->tau_g > 0.0) ? 1.0 / h->tau_g : 1.0;
    if (omega_g != 1.0) {
        double a2[3][3], A3[27], A4[81], A5[243], A6[729];
        for (int m = 0; m < 6; m++) a2[AB[m][0]][AB[m][1]] = a2[AB[m][1]][AB[m][0]] = a1[m];
        a1_recursion(a2, u, A3, A4, A5, A6);
        for (int k = 10; k < Q; k++) M[k] += (1.0 - omega_g) * a1_of_mode(k, a2, A3, A4, A5, A6);
    }
    /* body force, Guo in moment form (R13) */
    for (int a = 0; a < 3; a++) M[1 + a] += 0.5 * F[a];
    for (int m = 0; m < 6; m++) {
        int a = AB[m][0], b = AB[m][1];
        M[4 + m] += (1.0 - 0.5 * omega_h) * (u[a] * F[b] + u[b] * F[a]);
    }

    /* 6. noise on the non-conserved modes, Eq.8-9 */
    if (h->kT > 0.0) {
        uint32_t words[24];
        double r[Q];
        draw_site(h->seed, t, site, h->precision, words, r);
        double sq = sqrt(rho);
        for (int k = 4; k < Q; k++) {
            double om = (k <= 9) ? omega_h : omega_g;
            double sigma = sqrt(h->kT * om * (2.0 - om) * T_b[k] / cs2);
            M[k] += sq * sigma * r[k];
        }
    }

    /* 7. back-transform, Eq.10 */
    for (int i = 0; i < Q; i++) {
        double s = 0.0;
        for (int k = 0; k < Q; k++) s += M[k] * T_e[k][i] / T_b[k];
        fstar[i] = T_w[i] * s;
    }
}

/* BGK-FLBM, Eq.11, written in POPULATION space exactly as printed:
 *     f*_i = f_i^eq + (1 - omega) f_i^neq + w_i sum_k e_ki phi_k r_k / b_k,   f^neq = f - f^eq   (Eq.6 :85)
 * with ONE relaxation rate omega = 1/tau for every non-conserved mode, hence phi_k of Eq.9 (:99) at that omega
 * for all k = 4..26 (:95).  f^eq is not printed in Sec. II.A; reading R19: the same Hermite
 * equilibrium f^(0) of Eq.25 with Eq.20 that Reg-FLBM uses, so that the two models differ only in what happens
 * to the non-equilibrium part.  No body force in this model (the paper has none). */
static void collide_bgk(const rflbm_ref_t *h, const double g[Q], uint32_t site, uint64_t t, double fstar[Q])
{
    const double omega = 1.0 / h->tau;
    const double cs2 = 1.0 / 3.0;
    double rho = 0.0, u[3] = {0.0, 0.0, 0.0};
    for (int i = 0; i < Q; i++) rho += g[i];
    for (int a = 0; a < 3; a++) {
        for (int i = 0; i < Q; i++) u[a] += g[i] * (double)T_c[i][a];
        u[a] = u[a] / rho;
    }
    double feq[Q];
    rflbm_ref_equilibrium(rho, u, feq);
    for (int i = 0; i < Q; i++) fstar[i] = feq[i] + (1.0 - omega) * (g[i] - feq[i]);
    if (h->kT > 0.0) {
        uint32_t words[24];
        double r[Q], noise[Q];
        draw_site(h->seed, t, site, h->precision, words, r);
        for (int k = 0; k < Q; k++) noise[k] = 0.0;
        for (int k = 4; k < Q; k++) noise[k] = sqrt(rho * h->kT * omega * (2.0 - omega) * T_b[k] / cs2) * r[k];
        for (int i = 0; i < Q; i++) {
            double s = 0.0;
            for (int k = 4; k < Q; k++) s += noise[k] * T_e[k][i] / T_b[k];
            fstar[i] += T_w[i] * s;
        }
    }
}

/* single-site entry for the pin tests: BGK-FLBM */
int rflbm_ref_collide_site_bgk(const double g[Q], double tau, double kT, uint64_t seed, int precision,
                               uint32_t site, uint64_t t, double fstar[Q])
{
    build_tables();
    rflbm_ref_t h;
    memset(&h, 0, sizeof(h));
    h.tau = tau; h.kT = kT; h.seed = seed; h.precision = precision; h.model = REF_MODEL_BGK;
    collide_bgk(&h, g, site, t, fstar);
    return REF_OK;
}

/* single-site entry for the pin tests: collide with explicit parameters */
int rflbm_ref_collide_site(const double g[Q], double tau, double kT, uint64_t seed, int precision,
                           const double gacc[3], uint32_t site, uint64_t t, double fstar[Q])
{
    build_tables();
    rflbm_ref_t h;
    memset(&h, 0, sizeof(h));
    h.tau = tau; h.kT = kT; h.seed = seed; h.precision = precision;
    if (gacc) { h.g[0] = gacc[0]; h.g[1] = gacc[1]; h.g[2] = gacc[2]; }
    collide(&h, g, site, t, fstar);
    return REF_OK;
}

/* single-site entry with a ghost relaxation time (omega_g = 1/tau_g) */
int rflbm_ref_collide_site_ghost(const double g[Q], double tau, double tau_g, double kT, uint64_t seed, int precision,
                                 uint32_t site, uint64_t t, double fstar[Q])
{
    build_tables();
    rflbm_ref_t h;
    memset(&h, 0, sizeof(h));
    h.tau = tau; h.tau_g = tau_g; h.kT = kT; h.seed = seed; h.precision = precision;
    collide(&h, g, site, t, fstar);
    return REF_OK;
}

/* forward moment map m_k = sum_i e_ki f_i (Eq.4), for the pin tests */
void rflbm_ref_moments_of(const double f[Q], double m[Q])
{
    build_tables();
    for (int k = 0; k < Q; k++) {
        double s = 0.0;
        for (int i = 0; i < Q; i++) s += T_e[k][i] * f[i];
        m[k] = s;
    }
}

/* ------------------------------------------------------------------ time step */

static int wrap(int a, int n) { return (a < 0) ? a + n : (a >= n) ? a - n : a; }

static void step_once(rflbm_ref_t *h, int reverse_order)
{
    const int nx = h->nx, ny = h->ny, nz = h->nz;
    const size_t n = nsites(h);
    const double *S = h->S;
    double *S2 = h->S2;
    /* solid nodes keep their values */
    if (h->walls_z) {
        for (int i = 0; i < Q; i++)
            for (int zz = 0; zz < 2; zz++) {
                int z = zz ? nz - 1 : 0;
                size_t o = (size_t)i * n + (size_t)z * ny * nx;
                memcpy(S2 + o, S + o, sizeof(double) * (size_t)nx * ny);
            }
    }
#ifdef _OPENMP
#pragma omp parallel for num_threads(h->nthreads) schedule(static)
#endif
    for (int zi = 0; zi < nz; zi++) {
        int z = reverse_order ? nz - 1 - zi : zi;
        if (is_solid(h, z)) continue;
        for (int yi = 0; yi < ny; yi++) {
            int y = reverse_order ? ny - 1 - yi : yi;
            for (int xi = 0; xi < nx; xi++) {
                int x = reverse_order ? nx - 1 - xi : xi;
                size_t s = (size_t)x + (size_t)nx * ((size_t)y + (size_t)ny * z);
                double g[Q], fs[Q];
                for (int i = 0; i < Q; i++) g[i] = S[(size_t)i * n + s];      /* 1. */
                if (h->model == REF_MODEL_BGK) collide_bgk(h, g, (uint32_t)s, h->t, fs);
                else collide(h, g, (uint32_t)s, h->t, fs);                     /* 2.-7. */
                for (int i = 0; i < Q; i++) {                                  /* 8. stream, Eq.7 */
                    int xd = wrap(x + T_c[i][0], nx);
                    int yd = wrap(y + T_c[i][1], ny);
                    int zd = z + T_c[i][2];
                    if (h->walls_z) {
                        if (is_solid(h, zd)) {
                            /* halfway bounce-back (R12): reflected into the opposite direction at x */
                            S2[(size_t)T_opp[i] * n + s] = store_round(h, fs[i]);
                            continue;
                        }
                    } else {
                        zd = wrap(zd, nz);
                    }
                    size_t d = (size_t)xd + (size_t)nx * ((size_t)yd + (size_t)ny * zd);
                    S2[(size_t)i * n + d] = store_round(h, fs[i]);
                }
            }
        }
    }
    h->S = S2;
    h->S2 = (double *)S;
    h->t += 1;
}

int rflbm_ref_step(rflbm_ref_t *h, int nsteps)
{
    if (!h || nsteps < 0) return REF_EINVAL;
    if (!h->inited) return REF_ESTATE;
    for (int s = 0; s < nsteps; s++) step_once(h, 0);
    return REF_OK;
}

/* same step, sites visited in reverse order (order-independence pin P13) */
int rflbm_ref_step_reversed(rflbm_ref_t *h, int nsteps)
{
    if (!h || nsteps < 0) return REF_EINVAL;
    if (!h->inited) return REF_ESTATE;
    for (int s = 0; s < nsteps; s++) step_once(h, 1);
    return REF_OK;
}

/* ------------------------------------------------------------------ observables */

/* rho[N], u[3][N] from the current pre-collision state (step 2; u includes F/2).  Solid nodes: 0. */
int rflbm_ref_moments(rflbm_ref_t *h, double *rho, double *u)
{
    if (!h || !rho || !u) return REF_EINVAL;
    if (!h->inited) return REF_ESTATE;
    const size_t n = nsites(h);
    for (int z = 0; z < h->nz; z++)
        for (int y = 0; y < h->ny; y++)
            for (int x = 0; x < h->nx; x++) {
                size_t s = (size_t)x + (size_t)h->nx * ((size_t)y + (size_t)h->ny * z);
                if (is_solid(h, z)) { rho[s] = 0.0; u[s] = u[n + s] = u[2 * n + s] = 0.0; continue; }
                double r = 0.0, j[3] = {0.0, 0.0, 0.0};
                for (int i = 0; i < Q; i++) r += h->S[(size_t)i * n + s];
                for (int a = 0; a < 3; a++)
                    for (int i = 0; i < Q; i++) j[a] += h->S[(size_t)i * n + s] * (double)T_c[i][a];
                rho[s] = r;
                for (int a = 0; a < 3; a++) u[(size_t)a * n + s] = (j[a] + 0.5 * r * h->g[a]) / r;
            }
    return REF_OK;
}

/* Momentum-flux tensor the paper saves with its snapshots and uses for Table III (:260):
 * Pi_ab = a_0,ab^(2) + a_1,ab^(2) = sum_i f_i (c_ia c_ib - cs2 delta_ab)  (Eq.18 :150 + Eq.19 :153; the rho u u
 * terms cancel).  pi[6][N] in the order xx, yy, zz, xy, xz, yz (modes k = 4..9 of Table II); solid nodes: 0. */
int rflbm_ref_stress(rflbm_ref_t *h, double *pi)
{
    if (!h || !pi) return REF_EINVAL;
    if (!h->inited) return REF_ESTATE;
    static const int AB[6][2] = {{0, 0}, {1, 1}, {2, 2}, {0, 1}, {0, 2}, {1, 2}};
    const size_t n = nsites(h);
    for (int z = 0; z < h->nz; z++)
        for (size_t s = (size_t)z * h->nx * h->ny; s < (size_t)(z + 1) * h->nx * h->ny; s++)
            for (int m = 0; m < 6; m++) {
                double v = 0.0;
                if (!is_solid(h, z))
                    for (int i = 0; i < Q; i++)
                        v += h->S[(size_t)i * n + s] *
                             ((double)(T_c[i][AB[m][0]] * T_c[i][AB[m][1]]) - (AB[m][0] == AB[m][1] ? 1.0 / 3.0 : 0.0));
                pi[(size_t)m * n + s] = v;
            }
    return REF_OK;
}

/* out = { sum rho, sum rho u_x,y,z, mean u_x,y,z, var u_x,y,z } over fluid sites */
int rflbm_ref_diagnostics(rflbm_ref_t *h, double out[10])
{
    if (!h || !out) return REF_EINVAL;
    if (!h->inited) return REF_ESTATE;
    const size_t n = nsites(h);
    double *rho = (double *)malloc(sizeof(double) * n);
    double *u = (double *)malloc(sizeof(double) * 3 * n);
    if (!rho || !u) { free(rho); free(u); return REF_ENOMEM; }
    rflbm_ref_moments(h, rho, u);
    double mass = 0.0, P[3] = {0, 0, 0}, su[3] = {0, 0, 0}, suu[3] = {0, 0, 0};
    size_t nf = 0;
    for (int z = 0; z < h->nz; z++) {
        if (is_solid(h, z)) continue;
        for (size_t s = (size_t)z * h->nx * h->ny; s < (size_t)(z + 1) * h->nx * h->ny; s++) {
            mass += rho[s];
            for (int a = 0; a < 3; a++) {
                double ua = u[(size_t)a * n + s];
                P[a] += rho[s] * ua;
                su[a] += ua;
                suu[a] += ua * ua;
            }
            nf++;
        }
    }
    out[0] = mass;
    for (int a = 0; a < 3; a++) {
        out[1 + a] = P[a];
        out[4 + a] = su[a] / (double)nf;
        out[7 + a] = suu[a] / (double)nf - out[4 + a] * out[4 + a];
    }
    free(rho); free(u);
    return REF_OK;
}

int rflbm_ref_get_populations(rflbm_ref_t *h, double *f)
{
    if (!h || !f) return REF_EINVAL;
    if (!h->inited) return REF_ESTATE;
    memcpy(f, h->S, sizeof(double) * Q * nsites(h));
    return REF_OK;
}

int rflbm_ref_set_populations(rflbm_ref_t *h, const double *f, uint64_t step)
{
    if (!h || !f) return REF_EINVAL;
    size_t n = Q * nsites(h);
    for (size_t m = 0; m < n; m++) h->S[m] = store_round(h, f[m]);
    h->t = step;
    h->inited = 1;
    return REF_OK;
}

/* what the step would draw at `step`: words[24][N] (uint32), normals[23][N] (modes 4..26) */
int rflbm_ref_debug_rng(rflbm_ref_t *h, uint64_t step, uint32_t *words, double *normals)
{
    if (!h) return REF_EINVAL;
    const size_t n = nsites(h);
    for (size_t s = 0; s < n; s++) {
        uint32_t w[24];
        double r[Q];
        draw_site(h->seed, step, (uint32_t)s, h->precision, w, r);
        if (words) for (int m = 0; m < 24; m++) words[(size_t)m * n + s] = w[m];
        if (normals) for (int k = 4; k < Q; k++) normals[(size_t)(k - 4) * n + s] = r[k];
    }
    return REF_OK;
}
