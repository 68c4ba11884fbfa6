/*
 * vegas_oracle.c -- plain, slow, single-threaded CPU oracle for one Vegas iteration + grid refinement.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it.  It shares no source, header, table or constant
 * generator with the CUDA path under paper_2010_09341_b200/csrc/.
 *
 * What it computes and where each step is defined
 * -----------------------------------------------
 * The paper (refs [1,2] PAPER.md:L117-L118) only *names* the method:
 * Vegas importance sampling on an adaptive per-dimension grid where "every iteration informs the
 * subsequent run".  It prints no equation.  The arithmetic below is therefore the reading fixed in
 * SURVEY.md section 8.c (steps S1-S7, integrands I0-I4, readings R1-R17, restated in DESIGN.md) of
 * BASELINE.json:north_star.  The algorithm is followed step by step, in that notation; there is no
 * blocking, fusion or reordering.
 *
 *   S1  random stream   Philox4x32-10, key=(seed lo, seed hi), counter=(e lo, e hi, iteration, j)
 *   S2  map             exact integer bin rule  p=m*N, i=p>>B, frac=(p mod 2^B)/2^B ; x=fma(frac,wd,lo) ; J=prod g
 *   S3  integrand       I0 gauss_sym, I1 gauss_double, I2 genz_osc_peak (fp32), I3 lo_2to2, I4 toy_sum
 *   S4  weight          wf=(double)J*(double)f ; q=wf*wf
 *   S5  sums            S1=sum wf, S2=sum q, H[k][i_k]+=q      (Neumaier-compensated fp64)
 *   S6  estimate        I=S1/n ; V=(S2/n-I*I)/(n-1) ; sigma=sqrt(max(V,0))
 *   S7  refine(alpha)   3-point smoothing, ((1-r)/ln(1/r))^alpha damping, prefix sums, linear rebinning
 *
 * Parity pins (tests/test_oracle_*.py, all "-m 'not gpu'"): Philox known answers (P1), worked example
 * (P2, tests/golden/), closed-form integrals within 4 sigma (P3), invariants (P4), per-bin Gauss-Legendre
 * quadrature of the grid-mapped integrand for d<=2 (P5), exact-rational estimator and hand-checked refine
 * cases (P6), cos_f32 against fp64 cos (P7).  S7's *choice* of smoothing kernel and of prefix-sum
 * rebinning is fixed only by DESIGN.md readings R9/R12 ("parity unpinned" for that choice alone; the
 * arithmetic of the chosen form is pinned by P4/P6).
 *
 * Build:  gcc -O2 -std=c11 -ffp-contract=off -fno-fast-math -fPIC -shared vegas_oracle.c -lm
 * (-ffp-contract=off: every fused multiply-add below is an explicit fma()/fmaf() call.)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

enum { ORACLE_OK = 0, ORACLE_EINVAL = -1, ORACLE_ENOMEM = -3, ORACLE_ESTATE = -4,
       ORACLE_EUNSUPPORTED = -5, ORACLE_EGRID = -6 };
enum { ORACLE_FP64 = 0, ORACLE_FP32_EVAL = 1, ORACLE_FP64_U32 = 2 };
/* ORACLE_FP64_U32: fp64 arithmetic, one 32-bit Philox word per coordinate (B = 32): the extra stream mode of
 * DESIGN.md reading R3.  is_f64() is true for both fp64 modes. */
#define is_f64(c) ((c)->precision != ORACLE_FP32_EVAL)
#define ubits(c) ((c)->precision == ORACLE_FP64 ? 52 : ((c)->precision == ORACLE_FP64_U32 ? 32 : 23))
enum { ID_GAUSS_SYM = 0, ID_GAUSS_DOUBLE = 1, ID_GENZ_OSC_PEAK = 2, ID_LO_2TO2 = 3, ID_TOY_SUM = 4, ID_USER = 5, ID_LO_2TO2_TAB = 6 };
/* ID_USER: a user-supplied integrand f(x, dim, params) (the user writes the function of the
 * points); the tests compile the same C source with gcc that the CUDA side compiles at run time. */
typedef double (*oracle_user_fn)(const double *x, int dim, const double *params);

/* fl64(pi) = 3.141592653589793115997963... */
#define ORACLE_PI 0x1.921fb54442d18p+1

#define ORACLE_MAX_DIM 32
#define ORACLE_MAX_PARAMS 64

typedef struct oracle_ctx {
    int dim, nbins, integrand_id, precision;
    int n_params;
    double params[ORACLE_MAX_PARAMS];
    uint32_t iteration;   /* counter word 2 of S1; +1 per committed iteration */
    double *tab; int ntab;    /* ID_LO_2TO2_TAB: tabulated PDF G_j = g(x_j), knots uniform in ln x (oracle_set_table) */
    oracle_user_fn user_fn;   /* ID_USER: set by oracle_set_user_integrand before the first event */
    int uniform;          /* 1 after create/reset: table uses wd=fl(1/N) (S2, reading R6) */
    int have_hist;
    double *edges;        /* [dim][nbins+1] fp64 master edges E */
    double *hist;         /* [dim][nbins]   H of the last committed iteration */
    /* mapping table T[k][i]=(lo,wd,g), S2.  fp64 mode uses the d-arrays, fp32 mode the f-arrays. */
    double *lo_d, *wd_d, *g_d;
    float *lo_f, *wd_f, *g_f;
    double last_S1, last_S2;
    /* integrand constants, computed once from params with correctly rounded operations */
    double gC, ga2, gmu[2];                       /* I0 / I1 */
    float zphi, zc[ORACLE_MAX_DIM], zw[ORACLE_MAX_DIM];   /* I2 */
    double hs, hL, hcut, ha;                       /* I3 */
} oracle_ctx;

/* ------------------------------------------------------------------------------------------------
 * S1 -- Philox4x32-10 (Salmon et al., SC'11), exactly as published: multipliers 0xD2511F53 (word 0)
 * and 0xCD9E8D57 (word 2), Weyl key increments 0x9E3779B9 / 0xBB67AE85, ten rounds, round output
 * (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)).            [SURVEY 8.c S1, reading R2]
 * ---------------------------------------------------------------------------------------------- */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* S1 counter/key layout: key=(seed&0xFFFFFFFF, seed>>32); counter=(e&0xFFFFFFFF, e>>32, it, j). */
static void event_words(uint64_t seed, uint32_t it, uint64_t e, uint32_t j, uint32_t r[4])
{
    uint32_t ctr[4] = { (uint32_t)(e & 0xFFFFFFFFu), (uint32_t)(e >> 32), it, j };
    uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    oracle_philox4x32_10(ctr, key, r);
}

/* S1: the d mantissas of event e.  fp64 mode: coordinate k uses block j=k>>1, words a=2(k&1), a+1,
 * m=((r[a+1]<<32)+r[a])>>12 (52 bits).  fp32 mode: j=k>>2, m=r[k&3]>>9 (23 bits).   [reading R3] */
void oracle_mantissas(const oracle_ctx *c, uint64_t seed, uint32_t it, uint64_t e, uint64_t *m)
{
    uint32_t r[4];
    if (c->precision == ORACLE_FP64_U32) {                 /* m = r[k&3]: all 32 bits of one word */
        for (int k = 0; k < c->dim; ++k) {
            if ((k & 3) == 0) event_words(seed, it, e, (uint32_t)(k >> 2), r);
            m[k] = (uint64_t)r[k & 3];
        }
    } else if (c->precision == ORACLE_FP64) {
        for (int k = 0; k < c->dim; ++k) {
            if ((k & 1) == 0) event_words(seed, it, e, (uint32_t)(k >> 1), r);
            int a = 2 * (k & 1);
            m[k] = ((((uint64_t)r[a + 1]) << 32) | (uint64_t)r[a]) >> 12;
        }
    } else {
        for (int k = 0; k < c->dim; ++k) {
            if ((k & 3) == 0) event_words(seed, it, e, (uint32_t)(k >> 2), r);
            m[k] = (uint64_t)(r[k & 3] >> 9);
        }
    }
}

/* ------------------------------------------------------------------------------------------------
 * cos_f32 -- the specified single-precision cosine of integrand I2, valid |a|<=128.
 * Cody-Waite reduction by pi/2 in three fp32 pieces, Taylor polynomials, all in explicit fmaf.
 * ---------------------------------------------------------------------------------------------- */
float oracle_cos_f32(float a)
{
    const float K  = 0x1.45f306p-1f;     /* rnd32(2/pi) */
    const float C1 = 0x1.921fb6p+0f;     /* rnd32(pi/2) */
    const float C2 = -0x1.777a5cp-25f;   /* rnd32(pi/2 - C1) */
    const float C3 = -0x1.ee59dap-50f;   /* rnd32(pi/2 - C1 - C2) */
    float qf = rintf(a * K);
    float r = fmaf(qf, -C1, a);
    r = fmaf(qf, -C2, r);
    r = fmaf(qf, -C3, r);
    float z = r * r;
    /* cos r = 1 - z/2! + z^2/4! - z^3/6! + z^4/8! - z^5/10!   (Horner) */
    float pc = -0x1.27e4fcp-22f;                 /* rnd32(-1/3628800) */
    pc = fmaf(pc, z, 0x1.a01a02p-16f);           /* rnd32( 1/40320)   */
    pc = fmaf(pc, z, -0x1.6c16c2p-10f);          /* rnd32(-1/720)     */
    pc = fmaf(pc, z, 0x1.555556p-5f);            /* rnd32( 1/24)      */
    pc = fmaf(pc, z, -0.5f);
    pc = fmaf(pc, z, 1.0f);
    /* sin r = r + (z r)(-1/3! + z/5! - z^2/7! + z^3/9! - z^4/11!)   (Horner) */
    float ps = -0x1.ae6456p-26f;                 /* rnd32(-1/39916800) */
    ps = fmaf(ps, z, 0x1.71de3ap-19f);           /* rnd32( 1/362880)   */
    ps = fmaf(ps, z, -0x1.a01a02p-13f);          /* rnd32(-1/5040)     */
    ps = fmaf(ps, z, 0x1.111112p-7f);            /* rnd32( 1/120)      */
    ps = fmaf(ps, z, -0x1.555556p-3f);           /* rnd32(-1/6)        */
    float zr = z * r;
    float sn = fmaf(zr, ps, r);
    switch (((int)qf) & 3) {                     /* cos(q pi/2 + r) */
    case 0: return pc;
    case 1: return -sn;
    case 2: return -pc;
    default: return sn;
    }
}

void oracle_cos_f32_batch(const float *a, float *out, uint64_t n)
{
    for (uint64_t i = 0; i < n; ++i) out[i] = oracle_cos_f32(a[i]);
}

/* ------------------------------------------------------------------------------------------------
 * S2 -- mapping table.  Uniform grid (create/reset): E[k][i]=fl64(i/N), lo=rnd(E), wd=rnd(fl64(1/N)),
 * g=fl(N*wd).  Otherwise from the fp64 master edges: lo=rnd(E[i]), wd=rnd(fl64(E[i+1]-E[i])), g=fl(N*wd).
 * rnd = fp64 -> working precision.                                              [readings R5, R6]
 * ---------------------------------------------------------------------------------------------- */
static void rebuild_table(oracle_ctx *c)
{
    const int d = c->dim, N = c->nbins;
    for (int k = 0; k < d; ++k) {
        const double *E = c->edges + (size_t)k * (N + 1);
        for (int i = 0; i < N; ++i) {
            double wd = c->uniform ? (1.0 / (double)N) : (E[i + 1] - E[i]);
            size_t t = (size_t)k * N + i;
            c->lo_d[t] = E[i];
            c->wd_d[t] = wd;
            c->g_d[t] = (double)N * wd;
            c->lo_f[t] = (float)E[i];
            c->wd_f[t] = (float)wd;
            c->g_f[t] = (float)N * c->wd_f[t];
        }
    }
}

static void set_uniform(oracle_ctx *c)
{
    const int d = c->dim, N = c->nbins;
    for (int k = 0; k < d; ++k)
        for (int i = 0; i <= N; ++i)
            c->edges[(size_t)k * (N + 1) + i] = (i == N) ? 1.0 : (double)i / (double)N;
    c->uniform = 1;
    rebuild_table(c);
}

/* Integrand constants, one correctly rounded operation per step. */
static int setup_integrand(oracle_ctx *c)
{
    const double *p = c->params;
    switch (c->integrand_id) {
    case ID_GAUSS_SYM:      /* params {alpha, mu} */
    case ID_GAUSS_DOUBLE: { /* params {alpha, mu1, mu2} */
        int need = (c->integrand_id == ID_GAUSS_SYM) ? 2 : 3;
        if (c->n_params != need || !is_f64(c)) return ORACLE_EINVAL;
        double alpha = p[0];
        double b = alpha * sqrt(ORACLE_PI);        /* b = fl(alpha*fl(sqrt(pi))) */
        double C = 1.0;
        for (int k = 0; k < c->dim; ++k) C = C / b;
        c->gC = C;
        c->ga2 = 1.0 / (alpha * alpha);       /* a2 = fl(1/fl(alpha*alpha)) */
        c->gmu[0] = p[1];
        c->gmu[1] = (need == 3) ? p[2] : 0.0;
        return ORACLE_OK;
    }
    case ID_GENZ_OSC_PEAK: { /* params {phase_fraction, c_0..c_{d-1}}; fp32 only */
        if (c->n_params != 1 + c->dim || c->precision != ORACLE_FP32_EVAL) return ORACLE_EINVAL;
        c->zphi = (float)((2.0 * ORACLE_PI) * p[0]);
        for (int k = 0; k < c->dim; ++k) {
            float ck = (float)p[1 + k];
            c->zc[k] = ck;
            c->zw[k] = 1.0f / (ck * ck);
        }
        return ORACLE_OK;
    }
    case ID_LO_2TO2: { /* params {sqrt_s, sqrt_shat_min, cos_cut, pdf_a, pdf_b}; pdf_b fixed = 5 */
        if (c->n_params != 5 || c->dim != 3 || !is_f64(c)) return ORACLE_EINVAL;
        if (p[4] != 5.0) return ORACLE_EUNSUPPORTED;
        double s = p[0] * p[0];
        double smin = p[1] * p[1];
        double tau = smin / s;
        c->hs = s;
        c->hL = log(tau);
        c->hcut = p[2];
        c->ha = p[3];
        return ORACLE_OK;
    }
    case ID_LO_2TO2_TAB: { /* params {sqrt_s, sqrt_shat_min, cos_cut}; the PDF comes from oracle_set_table */
        if (c->n_params != 3 || c->dim != 3 || !is_f64(c)) return ORACLE_EINVAL;
        double s = p[0] * p[0];
        double smin = p[1] * p[1];
        c->hs = s;
        c->hL = log(smin / s);
        c->hcut = p[2];
        return ORACLE_OK;
    }
    case ID_TOY_SUM:
        if (c->n_params != 0) return ORACLE_EINVAL;
        return ORACLE_OK;
    case ID_USER:             /* params are handed to the user function as they are */
        if (!is_f64(c) || c->n_params > 16) return ORACLE_EINVAL;
        return ORACLE_OK;
    default:
        return ORACLE_EUNSUPPORTED;
    }
}

int oracle_create(oracle_ctx **out, int dim, int nbins, int integrand_id, const double *params,
                  int n_params, int precision)
{
    if (!out || dim < 1 || dim > ORACLE_MAX_DIM || nbins < 2 || n_params < 0 ||
        n_params > ORACLE_MAX_PARAMS || (n_params > 0 && !params))
        return ORACLE_EINVAL;
    if (precision != ORACLE_FP64 && precision != ORACLE_FP32_EVAL && precision != ORACLE_FP64_U32) return ORACLE_EINVAL;
    /* p=m*N must fit: N<2^12 with 52-bit m, N<2^9 with 23-bit m (S2) */
    if ((precision != ORACLE_FP32_EVAL && nbins >= 4096) || (precision == ORACLE_FP32_EVAL && nbins >= 512))
        return ORACLE_EINVAL;
    oracle_ctx *c = (oracle_ctx *)calloc(1, sizeof(oracle_ctx));
    if (!c) return ORACLE_ENOMEM;
    c->dim = dim; c->nbins = nbins; c->integrand_id = integrand_id; c->precision = precision;
    c->n_params = n_params;
    for (int i = 0; i < n_params; ++i) c->params[i] = params[i];
    int rc = setup_integrand(c);
    if (rc != ORACLE_OK) { free(c); return rc; }
    size_t cells = (size_t)dim * nbins;
    c->edges = (double *)calloc((size_t)dim * (nbins + 1), sizeof(double));
    c->hist = (double *)calloc(cells, sizeof(double));
    c->lo_d = (double *)calloc(cells, sizeof(double));
    c->wd_d = (double *)calloc(cells, sizeof(double));
    c->g_d = (double *)calloc(cells, sizeof(double));
    c->lo_f = (float *)calloc(cells, sizeof(float));
    c->wd_f = (float *)calloc(cells, sizeof(float));
    c->g_f = (float *)calloc(cells, sizeof(float));
    if (!c->edges || !c->hist || !c->lo_d || !c->wd_d || !c->g_d || !c->lo_f || !c->wd_f || !c->g_f)
        return ORACLE_ENOMEM;
    set_uniform(c);
    *out = c;
    return ORACLE_OK;
}

void oracle_destroy(oracle_ctx *c)
{
    if (!c) return;
    free(c->edges); free(c->hist); free(c->lo_d); free(c->wd_d); free(c->g_d);
    free(c->lo_f); free(c->wd_f); free(c->g_f); free(c->tab);
    free(c);
}

int oracle_reset(oracle_ctx *c)
{
    if (!c) return ORACLE_EINVAL;
    set_uniform(c);
    c->iteration = 0;
    c->have_hist = 0;
    return ORACLE_OK;
}

int oracle_set_iteration(oracle_ctx *c, uint32_t it) { if (!c) return ORACLE_EINVAL; c->iteration = it; return ORACLE_OK; }
uint32_t oracle_get_iteration(const oracle_ctx *c) { return c ? c->iteration : 0; }

int oracle_get_grid(const oracle_ctx *c, double *edges)
{
    if (!c || !edges) return ORACLE_EINVAL;
    memcpy(edges, c->edges, sizeof(double) * (size_t)c->dim * (c->nbins + 1));
    return ORACLE_OK;
}

int oracle_set_grid(oracle_ctx *c, const double *edges)
{
    if (!c || !edges) return ORACLE_EINVAL;
    const int d = c->dim, N = c->nbins;
    for (int k = 0; k < d; ++k) {
        const double *E = edges + (size_t)k * (N + 1);
        if (E[0] != 0.0 || E[N] != 1.0) return ORACLE_EGRID;
        for (int i = 0; i < N; ++i)
            if (!(E[i] < E[i + 1])) return ORACLE_EGRID;
    }
    memcpy(c->edges, edges, sizeof(double) * (size_t)d * (N + 1));
    c->uniform = 0;
    rebuild_table(c);
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------------
 * S3 -- integrands, normative evaluation order.
 * ---------------------------------------------------------------------------------------------- */
/* Tabulated PDF: M knots uniform in ln x.  x = tau^v, so ln x = v L is linear in v: knot j sits at
 * v_j = 1 - j/(M-1), i.e. G_0 = g(tau) (v = 1) ... G_{M-1} = g(1) (v = 0).
 * u = (1 - v)(M - 1); j = floor(u) clamped to [1, M-3]; s = u - j; four-point Lagrange (cubic) interpolation
 *   w0 = -s(s-1)(s-2)/6, w1 = (s+1)(s-1)(s-2)/2, w2 = -(s+1)s(s-2)/2, w3 = (s+1)s(s-1)/6,
 *   g = ((w0 G[j-1] + w1 G[j]) + w2 G[j+1]) + w3 G[j+2]          (plain products and sums, that order). */
static double tab_interp(const double *G, int M, double v)
{
    double u = (1.0 - v) * (double)(M - 1);
    int j = (int)floor(u);
    if (j < 1) j = 1;
    if (j > M - 3) j = M - 3;
    double s = u - (double)j;
    double sp = s + 1.0, sm1 = s - 1.0, sm2 = s - 2.0;
    double w0 = -((s * sm1) * sm2) / 6.0;
    double w1 = ((sp * sm1) * sm2) / 2.0;
    double w2 = -((sp * s) * sm2) / 2.0;
    double w3 = ((sp * s) * sm1) / 6.0;
    return ((w0 * G[j - 1] + w1 * G[j]) + w2 * G[j + 1]) + w3 * G[j + 2];
}

static double eval_fp64(const oracle_ctx *c, const double *x, int *pass_out)
{
    const int d = c->dim;
    *pass_out = 1;
    switch (c->integrand_id) {
    case ID_GAUSS_SYM: {      /* f = prod_k exp(-(x_k-mu)^2/alpha^2)/(alpha sqrt(pi))   BASELINE.json configs[0] */
        double s = 0.0;
        for (int k = 0; k < d; ++k) { double dx = x[k] - c->gmu[0]; s = fma(dx, dx, s); }
        return c->gC * exp(-(s * c->ga2));
    }
    case ID_GAUSS_DOUBLE: {   /* f = 1/2 C [exp(-s1 a2) + exp(-s2 a2)]                  BASELINE.json configs[1] */
        double s1 = 0.0, s2 = 0.0;
        for (int k = 0; k < d; ++k) { double dx = x[k] - c->gmu[0]; s1 = fma(dx, dx, s1); }
        for (int k = 0; k < d; ++k) { double dx = x[k] - c->gmu[1]; s2 = fma(dx, dx, s2); }
        double e1 = exp(-(s1 * c->ga2));
        double e2 = exp(-(s2 * c->ga2));
        return (0.5 * c->gC) * (e1 + e2);
    }
    case ID_LO_2TO2: {        /* BASELINE.json configs[4], reading R15 */
        const double v1 = x[0], v2 = x[1], v3 = x[2];
        const double L = c->hL, s = c->hs;
        double cth = fma(2.0, v3, -1.0);
        int pass = ((v1 + v2) < 1.0) && (fabs(cth) < c->hcut);
        *pass_out = pass;
        if (!pass) return 0.0;
        double x1 = exp(v1 * L);
        double x2 = exp(v2 * L);
        double x12 = x1 * x2;
        double shat = x12 * s;
        double that = (-0.5 * shat) * (1.0 - cth);
        double uhat = (-0.5 * shat) * (1.0 + cth);
        double ME = (shat * shat + uhat * uhat) / (that * that);
        double y1 = 1.0 - x1, y2 = 1.0 - x2;
        double y1p5 = ((y1 * y1) * (y1 * y1)) * y1;
        double y2p5 = ((y2 * y2) * (y2 * y2)) * y2;
        double g1 = exp(-c->ha * (v1 * L)) * y1p5;      /* x1^-a (1-x1)^5 */
        double g2 = exp(-c->ha * (v2 * L)) * y2p5;
        double flux = 1.0 / (2.0 * shat);
        double Jac = (x12 * (L * L)) * 2.0;             /* |d(x1,x2,cos)/d(v1,v2,v3)| */
        return (((g1 * g2) * ME) * flux) * Jac;
    }
    case ID_LO_2TO2_TAB: {    /* I3 with g(x) interpolated from a table (PDFFlow-style lookup,
                               * PAPER.md:L33, L49; a synthetic table stands in for a PDF grid) */
        const double v1 = x[0], v2 = x[1], v3 = x[2];
        const double L = c->hL, s = c->hs;
        double cth = fma(2.0, v3, -1.0);
        int pass = ((v1 + v2) < 1.0) && (fabs(cth) < c->hcut);
        *pass_out = pass;
        if (!pass) return 0.0;
        if (!c->tab) return NAN;
        double x1 = exp(v1 * L);
        double x2 = exp(v2 * L);
        double x12 = x1 * x2;
        double shat = x12 * s;
        double that = (-0.5 * shat) * (1.0 - cth);
        double uhat = (-0.5 * shat) * (1.0 + cth);
        double ME = (shat * shat + uhat * uhat) / (that * that);
        double g1 = tab_interp(c->tab, c->ntab, v1);
        double g2 = tab_interp(c->tab, c->ntab, v2);
        double flux = 1.0 / (2.0 * shat);
        double Jac = (x12 * (L * L)) * 2.0;
        return (((g1 * g2) * ME) * flux) * Jac;
    }
    case ID_TOY_SUM: {        /* PAPER.md:L72-L73  tf.reduce_sum(xarr, axis=1) */
        double f = 0.0;
        for (int k = 0; k < d; ++k) f = f + x[k];
        return f;
    }
    case ID_USER:
        return c->user_fn ? c->user_fn(x, d, c->params) : NAN;
    default:
        return NAN;
    }
}

static float eval_fp32(const oracle_ctx *c, const float *x)
{
    const int d = c->dim;
    switch (c->integrand_id) {
    case ID_GENZ_OSC_PEAK: {  /* f = cos(phi + sum c_k x_k) / prod (c_k^-2 + (x_k-1/2)^2)   BASELINE.json configs[3] */
        float arg = c->zphi, Q = 1.0f;
        for (int k = 0; k < d; ++k) {
            arg = fmaf(c->zc[k], x[k], arg);
            float dx = x[k] - 0.5f;
            float pk = fmaf(dx, dx, c->zw[k]);
            Q = Q * pk;
        }
        return oracle_cos_f32(arg) / Q;
    }
    case ID_TOY_SUM: {
        float f = 0.0f;
        for (int k = 0; k < d; ++k) f = f + x[k];
        return f;
    }
    default:
        return NAN;
    }
}

/* ------------------------------------------------------------------------------------------------
 * S2-S4 for one event given its d mantissas.  Outputs: bins, x (as double), J (as double), f (as
 * double), wf (S4), pass flag (I3's cut; 1 elsewhere).
 * ---------------------------------------------------------------------------------------------- */
static void map_eval(const oracle_ctx *c, const uint64_t *m, int32_t *bins, double *xo, double *jo,
                     double *fo, double *wfo, int *passo)
{
    const int d = c->dim, N = c->nbins;
    if (is_f64(c)) {
        const int B = ubits(c);                                   /* 52, or 32 in the 32-bit-uniform mode */
        double x[ORACLE_MAX_DIM];
        double J = 0.0;
        for (int k = 0; k < d; ++k) {
            uint64_t p = m[k] * (uint64_t)N;                       /* exact: m<2^B<=2^52, N<2^12 */
            int i = (int)(p >> B);
            double frac = ldexp((double)(p & ((1ull << B) - 1)), -B);     /* exact */
            size_t t = (size_t)k * N + i;
            x[k] = fma(frac, c->wd_d[t], c->lo_d[t]);
            J = (k == 0) ? c->g_d[t] : J * c->g_d[t];
            bins[k] = i;
            xo[k] = x[k];
        }
        int pass;
        double f = eval_fp64(c, x, &pass);
        *jo = J; *fo = f; *wfo = J * f; *passo = pass;
    } else {
        float x[ORACLE_MAX_DIM];
        float J = 0.0f;
        for (int k = 0; k < d; ++k) {
            uint32_t p = (uint32_t)m[k] * (uint32_t)N;             /* exact: m<2^23, N<2^9 */
            int i = (int)(p >> 23);
            float frac = ldexpf((float)(p & ((1u << 23) - 1)), -23);      /* exact */
            size_t t = (size_t)k * N + i;
            x[k] = fmaf(frac, c->wd_f[t], c->lo_f[t]);
            J = (k == 0) ? c->g_f[t] : J * c->g_f[t];
            bins[k] = i;
            xo[k] = (double)x[k];
        }
        float f = eval_fp32(c, x);
        *jo = (double)J; *fo = (double)f; *wfo = (double)J * (double)f; *passo = 1;
    }
}

/* Per-event dump (parity hook): events first..first+count-1 of the current iteration counter. */
int oracle_events(const oracle_ctx *c, uint64_t first, uint32_t count, uint64_t seed, int32_t *bins,
                  double *x, double *jac, double *f, double *wf, int32_t *pass)
{
    if (!c) return ORACLE_EINVAL;
    uint64_t m[ORACLE_MAX_DIM];
    int32_t b[ORACLE_MAX_DIM];
    double xx[ORACLE_MAX_DIM];
    for (uint32_t n = 0; n < count; ++n) {
        double J, fv, w; int ps;
        oracle_mantissas(c, seed, c->iteration, first + n, m);
        map_eval(c, m, b, xx, &J, &fv, &w, &ps);
        for (int k = 0; k < c->dim; ++k) {
            if (bins) bins[(size_t)n * c->dim + k] = b[k];
            if (x) x[(size_t)n * c->dim + k] = xx[k];
        }
        if (jac) jac[n] = J;
        if (f) f[n] = fv;
        if (wf) wf[n] = w;
        if (pass) pass[n] = ps;
    }
    return ORACLE_OK;
}

/* S2-S4 at caller-chosen mantissas (quadrature pin P5): m is [count][dim]. */
int oracle_map_eval(const oracle_ctx *c, const uint64_t *m, uint32_t count, int32_t *bins, double *x,
                    double *jac, double *f)
{
    if (!c || !m) return ORACLE_EINVAL;
    int32_t b[ORACLE_MAX_DIM];
    double xx[ORACLE_MAX_DIM];
    const uint64_t lim = 1ull << ubits(c);
    for (uint32_t n = 0; n < count; ++n) {
        double J, fv, w; int ps;
        for (int k = 0; k < c->dim; ++k)
            if (m[(size_t)n * c->dim + k] >= lim) return ORACLE_EINVAL;
        map_eval(c, m + (size_t)n * c->dim, b, xx, &J, &fv, &w, &ps);
        for (int k = 0; k < c->dim; ++k) {
            if (bins) bins[(size_t)n * c->dim + k] = b[k];
            if (x) x[(size_t)n * c->dim + k] = xx[k];
        }
        if (jac) jac[n] = J;
        if (f) f[n] = fv;
    }
    return ORACLE_OK;
}

/* S5: Neumaier-compensated accumulation (sum s, running compensation c; value = s + c). */
static inline void neumaier_add(double *s, double *c, double x)
{
    double t = *s + x;
    if (fabs(*s) >= fabs(x)) *c += (*s - t) + x;
    else                     *c += (x - t) + *s;
    *s = t;
}

/* S1-S5 over the event range [first, first+count) of the current iteration counter.  Does not touch
 * the context.  sums[4] = {S1.s, S1.c, S2.s, S2.c}; hist_s/hist_c = [dim][nbins] sum and compensation
 * (caller-zeroed or not: they are overwritten); npass = number of events passing I3's cut.
 * A harness may run disjoint ranges on several threads and add the pieces (events are counter-indexed,
 * so the real-number sums do not depend on the split). */
int oracle_iterate_range(const oracle_ctx *c, uint64_t first, uint64_t count, uint64_t seed,
                         double *sums, double *hist_s, double *hist_c, uint64_t *npass)
{
    if (!c || !sums || !hist_s || !hist_c) return ORACLE_EINVAL;
    const int d = c->dim, N = c->nbins;
    uint64_t m[ORACLE_MAX_DIM];
    int32_t b[ORACLE_MAX_DIM];
    double xx[ORACLE_MAX_DIM];
    double s1 = 0.0, c1 = 0.0, s2 = 0.0, c2 = 0.0;
    uint64_t np = 0;
    memset(hist_s, 0, sizeof(double) * (size_t)d * N);
    memset(hist_c, 0, sizeof(double) * (size_t)d * N);
    for (uint64_t e = first; e < first + count; ++e) {
        double J, f, wf; int ps;
        oracle_mantissas(c, seed, c->iteration, e, m);
        map_eval(c, m, b, xx, &J, &f, &wf, &ps);
        double q = wf * wf;                                   /* S4 */
        neumaier_add(&s1, &c1, wf);                           /* S5 */
        neumaier_add(&s2, &c2, q);
        for (int k = 0; k < d; ++k) {
            size_t t = (size_t)k * N + b[k];
            neumaier_add(&hist_s[t], &hist_c[t], q);
        }
        np += (uint64_t)ps;
    }
    sums[0] = s1; sums[1] = c1; sums[2] = s2; sums[3] = c2;
    if (npass) *npass = np;
    return ORACLE_OK;
}

/* S6 from the total sums; stores H, advances the iteration counter. */
int oracle_commit(oracle_ctx *c, uint64_t n_events, double S1, double S2, const double *hist,
                  double *integral, double *error)
{
    if (!c || !hist || !integral || !error || n_events < 2) return ORACLE_EINVAL;
    double n = (double)n_events;
    double I = S1 / n;
    double V = (S2 / n - I * I) / (n - 1.0);
    *integral = I;
    *error = sqrt(V > 0.0 ? V : 0.0);
    memcpy(c->hist, hist, sizeof(double) * (size_t)c->dim * c->nbins);
    c->have_hist = 1;
    c->last_S1 = S1; c->last_S2 = S2;
    c->iteration += 1;
    return ORACLE_OK;
}

/* One whole iteration, single-threaded: S1-S6. */
int oracle_iterate(oracle_ctx *c, uint64_t n_events, uint64_t seed, double *integral, double *error,
                   double *hist)
{
    if (!c || !integral || !error || n_events < 2) return ORACLE_EINVAL;
    size_t cells = (size_t)c->dim * c->nbins;
    double *hs = (double *)malloc(sizeof(double) * cells);
    double *hc = (double *)malloc(sizeof(double) * cells);
    if (!hs || !hc) { free(hs); free(hc); return ORACLE_ENOMEM; }
    double sums[4];
    int rc = oracle_iterate_range(c, 0, n_events, seed, sums, hs, hc, NULL);
    if (rc == ORACLE_OK) {
        for (size_t t = 0; t < cells; ++t) hs[t] = hs[t] + hc[t];
        rc = oracle_commit(c, n_events, sums[0] + sums[1], sums[2] + sums[3], hs, integral, error);
        if (rc == ORACLE_OK && hist) memcpy(hist, hs, sizeof(double) * cells);
    }
    free(hs); free(hc);
    return rc;
}

int oracle_last_sums(const oracle_ctx *c, double *S1, double *S2)
{
    if (!c || !c->have_hist) return ORACLE_ESTATE;
    if (S1) *S1 = c->last_S1;
    if (S2) *S2 = c->last_S2;
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------------
 * S7 -- refine(alpha): the classic Vegas grid adaptation (Lepage), per dimension,
 * fp64, from the histogram of the last committed iteration.  Readings R9-R12.
 * ---------------------------------------------------------------------------------------------- */
int oracle_refine(oracle_ctx *c, double alpha)
{
    if (!c || !(alpha >= 0.0)) return ORACLE_EINVAL;
    if (!c->have_hist) return ORACLE_ESTATE;
    const int d = c->dim, N = c->nbins;
    double *newE = (double *)malloc(sizeof(double) * (size_t)d * (N + 1));
    double *s = (double *)malloc(sizeof(double) * N);
    double *mm = (double *)malloc(sizeof(double) * N);
    double *cum = (double *)malloc(sizeof(double) * (N + 1));
    if (!newE || !s || !mm || !cum) { free(newE); free(s); free(mm); free(cum); return ORACLE_ENOMEM; }
    memcpy(newE, c->edges, sizeof(double) * (size_t)d * (N + 1));
    int rc = ORACLE_OK;
    for (int k = 0; k < d; ++k) {
        const double *h = c->hist + (size_t)k * N;
        const double *E = c->edges + (size_t)k * (N + 1);
        double *En = newE + (size_t)k * (N + 1);
        /* step 1: nothing to adapt to */
        double tot = 0.0;
        for (int i = 0; i < N; ++i) tot += h[i];
        if (!(tot > 0.0) || !isfinite(tot)) continue;
        /* step 2: 3-point smoothing, 2-point ends */
        s[0] = (h[0] + h[1]) / 2.0;
        s[N - 1] = (h[N - 2] + h[N - 1]) / 2.0;
        for (int i = 1; i < N - 1; ++i) s[i] = (h[i - 1] + h[i] + h[i + 1]) / 3.0;
        /* step 3: normalise */
        double ssum = 0.0;
        for (int i = 0; i < N; ++i) ssum += s[i];
        /* step 4: damping m_i = ((1-r)/ln(1/r))^alpha */
        for (int i = 0; i < N; ++i) {
            double r = s[i] / ssum;
            if (r <= 0.0) mm[i] = 0.0;
            else if (r >= 1.0) mm[i] = 1.0;
            else mm[i] = pow((1.0 - r) / (-log(r)), alpha);
        }
        /* step 5: prefix sums */
        cum[0] = 0.0;
        for (int i = 0; i < N; ++i) cum[i + 1] = cum[i] + mm[i];
        double delta = cum[N] / (double)N;
        /* step 6: N-1 new interior edges by linear interpolation inside old bins */
        En[0] = 0.0; En[N] = 1.0;
        int i = 0;
        for (int j = 1; j < N; ++j) {
            double t = (double)j * delta;
            while (i < N - 1 && !(cum[i + 1] >= t && mm[i] > 0.0)) ++i;
            En[j] = E[i] + ((t - cum[i]) / mm[i]) * (E[i + 1] - E[i]);
        }
        /* step 7: must stay strictly increasing */
        for (int j = 0; j < N; ++j)
            if (!(En[j] < En[j + 1])) rc = ORACLE_EGRID;
    }
    if (rc == ORACLE_OK) {
        memcpy(c->edges, newE, sizeof(double) * (size_t)d * (N + 1));
        c->uniform = 0;
        rebuild_table(c);
        memset(c->hist, 0, sizeof(double) * (size_t)d * N);
        c->have_hist = 0;
    }
    free(newE); free(s); free(mm); free(cum);
    return rc;
}

/* Table accessor for tests (S2 pins): fills lo, wd, g as doubles, [dim][nbins]. */
int oracle_get_table(const oracle_ctx *c, double *lo, double *wd, double *g)
{
    if (!c) return ORACLE_EINVAL;
    size_t cells = (size_t)c->dim * c->nbins;
    for (size_t t = 0; t < cells; ++t) {
        if (is_f64(c)) {
            if (lo) lo[t] = c->lo_d[t];
            if (wd) wd[t] = c->wd_d[t];
            if (g) g[t] = c->g_d[t];
        } else {
            if (lo) lo[t] = (double)c->lo_f[t];
            if (wd) wd[t] = (double)c->wd_f[t];
            if (g) g[t] = (double)c->g_f[t];
        }
    }
    return ORACLE_OK;
}

/* Integrand constants accessor for the worked-example pin P2: out[0]=C, out[1]=a2 (I0/I1). */
int oracle_get_gauss_consts(const oracle_ctx *c, double *out)
{
    if (!c || !out) return ORACLE_EINVAL;
    out[0] = c->gC; out[1] = c->ga2;
    return ORACLE_OK;
}

/*
 * run_integration (the combination formula is paper-silent: DESIGN.md reading R18, the classic
 * Vegas inverse-variance average of the cited references).
 *   w_i = 1/sigma_i^2 ; mean = (sum_i w_i I_i)/(sum_i w_i) ; error = 1/sqrt(sum_i w_i) ;
 *   chi2/dof = (sum_i w_i (I_i - mean)^2)/(n - 1)    (0 for n = 1)
 * Iterations whose sigma is zero or not finite carry no weight; if none does: plain average, error 0.
 */
int oracle_combine(int n, const double *I, const double *sigma, double *mean, double *err, double *chi2_dof)
{
    if (n < 1 || !I || !sigma || !mean || !err) return ORACLE_EINVAL;
    long double sum_w = 0.0L, sum_wi = 0.0L, sum_plain = 0.0L;
    int used = 0;
    for (int i = 0; i < n; ++i) {
        sum_plain += (long double)I[i];
        if (sigma[i] > 0.0 && isfinite(sigma[i]) && isfinite(I[i])) {
            long double w = 1.0L / ((long double)sigma[i] * (long double)sigma[i]);
            sum_w += w;
            sum_wi += w * (long double)I[i];
            ++used;
        }
    }
    if (used == 0) {
        *mean = (double)(sum_plain / n);
        *err = 0.0;
        if (chi2_dof) *chi2_dof = 0.0;
        return ORACLE_OK;
    }
    long double m = sum_wi / sum_w, chi2 = 0.0L;
    for (int i = 0; i < n; ++i)
        if (sigma[i] > 0.0 && isfinite(sigma[i]) && isfinite(I[i])) {
            long double w = 1.0L / ((long double)sigma[i] * (long double)sigma[i]);
            chi2 += w * ((long double)I[i] - m) * ((long double)I[i] - m);
        }
    *mean = (double)m;
    *err = (double)(1.0L / sqrtl(sum_w));
    if (chi2_dof) *chi2_dof = (n > 1) ? (double)(chi2 / (n - 1)) : 0.0;
    return ORACLE_OK;
}

/* ID_USER: the function evaluated in S3. */
int oracle_set_user_integrand(oracle_ctx *c, oracle_user_fn fn)
{
    if (!c || !fn || c->integrand_id != ID_USER) return ORACLE_EINVAL;
    c->user_fn = fn;
    return ORACLE_OK;
}

/* ID_LO_2TO2_TAB: the tabulated PDF (M >= 4 values, copied). */
int oracle_set_table(oracle_ctx *c, const double *values, int n)
{
    if (!c || !values || n < 4 || n > 4096) return ORACLE_EINVAL;
    double *t = (double *)malloc(sizeof(double) * (size_t)n);
    if (!t) return ORACLE_ENOMEM;
    memcpy(t, values, sizeof(double) * (size_t)n);
    free(c->tab);
    c->tab = t;
    c->ntab = n;
    return ORACLE_OK;
}

/* the interpolation alone, for its pins */
double oracle_tab_interp(const double *values, int n, double v) { return tab_interp(values, n, v); }
