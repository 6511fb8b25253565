/*
 * gn_oracle.c -- CPU ORACLE for the geometric-network simulation step.  TEST INFRASTRUCTURE.
 *
 * Plain, slow, obviously-correct C written from the paper (/root/reference/PAPER.md, Buibas &
 * Silva, arxiv 0908.3934) and from DESIGN.md's readings where the paper is silent.  It shares no
 * code, header, table or helper with the CUDA library and is imported only by tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
 *
 * What it computes (one call of orc_step = the paper's "advance the network by dt",
 * PAPER.md:68-71 eq. 5), for every vertex j, all reads being of the state at step t:
 *
 *   1. input     I_fx = sum over in-edges k->j with raster[t - delay_kj][k] = 1 of w_fx_kj
 *                (eq. 30's sum; kept as a delay ring, slot t mod D, read and zeroed),
 *                plus a Bernoulli kick from a counter generator (BASELINE.json's Poisson drive,
 *                injected like an arriving event, reading #12).  The user control U_j(t)
 *                (eq. 7) is an optional constant current inside eq. 28's bracket.
 *   2. detect    fired = (refr == 0) and (V >= v_peak)                   PAPER.md:316 eq. 31
 *   3. update    forward Euler (eq. 19) of the Izhikevich simple model with hard
 *                reset (eq. 24) and the PSC term +r(t) (eq. 28);
 *                absolute refractory hold (reading #6)
 *   4. PSC       r' = r (1 - dt/tau_s) + I                               PAPER.md:283-286 eq. 26
 *                or, for a class with psc_alpha != 0, the alpha-function of PAPER.md:288-312
 *                eq. 27, 29, 30 with a = 1/tau_s:  r' = r + dt p,  p' = p + dt (-a^2 r - 2a p) + I
 *                (the arriving weight is an impulse on p: eq. 27's p(t+) = p(t) + w, reading #4)
 *                A class with model = 1 is a Hodgkin-Huxley vertex instead ("states {v, m, n, h}", dt on the
 *                order of 0.03 ms; the paper's second benchmarked model).  The paper prints no equations
 *                for it: they are the textbook ones (Hodgkin & Huxley 1952 in the modern sign convention), restated
 *                at orc_vertex_hh_fp64 below, forward Euler (eq. 19) like everything else; no reset, the
 *                refractory counter is only the detection dead time that makes one action potential one event.
 *   5. calcium   c' = c (1 - dt/tau_c) + ca_jump * fired                 PAPER.md:364 H_c
 *   6. record    raster[t][j] = fired; deliver: every out-edge (j->m, w_fx, delay) of a fired j
 *                adds w_fx to ring[(t + delay) mod D][m]
 *   7. observe   frame mean of c' over obs_stride steps, z = n*mean + b + gamma*N(0,1)
 *                                                                        PAPER.md:370-374
 *
 * Two arithmetic modes:
 *   mode 0  fp64 -- the definition: all real state in double.
 *   mode 1  fp32-faithful -- every value binary32, one correctly rounded operation at a time in
 *           the written order, fmaf only where written.  Compile with -ffp-contract=off.
 * Delivery, the ring, the drive decision and the raster are pure integer in both modes.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): Philox known-answer vectors; fixed points and
 * closed forms of the update; Hodgkin-Huxley: textbook rate values and gating steady states at rest, the resting
 * fixed point, one action potential per supra-threshold pulse, the textbook firing rate at 10 uA/cm^2, orc_exp32 against
 * libm; geometric decay of r and c; the alpha-function PSC against the matrix
 * power of its 2x2 Euler map, its exact discrete integral w tau^2 and w t e^(-at); chain arrival steps; event-count and
 * fixed-point-mass conservation; the pure-Python pull definition (oracle/pull_definition.py) on
 * <= 10-node graphs; the implementation-free ring-content definition; noise statistics.
 * Parity unpinned: none of the functions below; the chaotic tail beyond the first fp32/fp64
 * raster divergence is unpinned against fp64 by nature.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC -o libgn_oracle.so gn_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------------------------------
 * Counter-based generator: Philox4x32-10 (Salmon, Moraes, Dror, Shaw, "Parallel random numbers:
 * as easy as 1, 2, 3", SC'11), written from its published description.  DESIGN.md reading #13.
 * ---------------------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
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

enum { ORC_STREAM_DRIVE = 5, ORC_STREAM_NOISE = 6 };

/* The 32-bit word of vertex j at index `idx` (a step or a frame) on `stream`:
 * counter = { j / 4, idx low, idx high, stream }, key = { seed low, seed high }, word j mod 4. */
uint32_t orc_word(uint64_t seed, uint32_t stream, uint32_t j, uint64_t idx)
{
    uint32_t ctr[4] = { j >> 2, (uint32_t)idx, (uint32_t)(idx >> 32), stream };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t out[4];
    orc_philox4x32_10(ctr, key, out);
    return out[j & 3];
}

/* Standard normal for (vertex j, frame): Box-Muller on two words of the vertex group's block.
 * Vertices j mod 4 in {0,1} share words (x0,x1), {2,3} share (x2,x3); even j takes the cosine
 * branch, odd j the sine branch.  u_a = (k + 1/2) 2^-23 in (0,1) from the top 23 bits, u_b = k 2^-24
 * in [0,1) from the top 24 bits (both exact in binary32 as well as in double). */
double orc_gauss(uint64_t seed, uint32_t j, uint64_t frame)
{
    uint32_t ctr[4] = { j >> 2, (uint32_t)frame, (uint32_t)(frame >> 32), ORC_STREAM_NOISE };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t x[4];
    orc_philox4x32_10(ctr, key, x);
    uint32_t xa = x[(j & 2)], xb = x[(j & 2) + 1];
    double ua = ((double)(xa >> 9) + 0.5) * (1.0 / 8388608.0);
    double ub = (double)(xb >> 8) * (1.0 / 16777216.0);
    double rad = sqrt(-2.0 * log(ua));
    double ang = 6.283185307179586476925286766559 * ub;
    return (j & 1) ? rad * sin(ang) : rad * cos(ang);
}

/* ------------------------------------------------------------------------------------------
 * Create-time quantities (each one a function so a test can pin it alone)
 * ---------------------------------------------------------------------------------------- */

/* PAPER.md:251 eq. 25, tau_ij = |x_i - x_j| / s, in whole steps: max(1, ceil(dist/(speed*dt))),
 * evaluated in double from the fp32 positions (reading #7). */
uint32_t orc_delay_steps(const float *xi, const float *xj, uint32_t dim, float speed, float dt_ms)
{
    double d2 = 0.0;
    for (uint32_t k = 0; k < dim; ++k) {
        double d = (double)xi[k] - (double)xj[k];
        d2 = d2 + d * d;
    }
    double steps = ceil(sqrt(d2) / ((double)speed * (double)dt_ms));
    if (steps < 1.0) steps = 1.0;
    if (steps > 4294967295.0) steps = 4294967295.0;
    return (uint32_t)steps;
}

/* int32 fixed point with 16 fractional bits: rint(w * 2^16), ties to even (BASELINE.json). */
int64_t orc_quantise(float w)
{
    return (int64_t)nearbyint((double)w * 65536.0);
}

/* Bernoulli(rate*dt) as an unsigned 32-bit threshold: floor(((rate*dt)*1e-3)*2^32), in double. */
uint32_t orc_drive_threshold(float rate_hz, float dt_ms)
{
    double p = (((double)rate_hz * (double)dt_ms) * 1e-3) * 4294967296.0;
    if (!(p > 0.0)) return 0;
    if (p >= 4294967295.0) return 4294967295u;
    return (uint32_t)floor(p);
}

/* 1 - dt/tau in double (the fp32 mode rounds it once to float). */
double orc_keep(float dt_ms, float tau_ms)
{
    return 1.0 - (double)dt_ms / (double)tau_ms;
}

uint32_t orc_refractory_steps(float refractory_ms, float dt_ms)
{
    double r = nearbyint((double)refractory_ms / (double)dt_ms);
    return r > 0.0 ? (uint32_t)r : 0u;
}

/* ------------------------------------------------------------------------------------------
 * Hodgkin-Huxley vertex class (the equations are the textbook ones, the paper
 * prints none):
 *     C dV/dt = -g_na m^3 h (V - e_na) - g_k n^4 (V - e_k) - g_l (V - e_l) + r + U
 *     dx/dt   = alpha_x(V) (1 - x) - beta_x(V) x                      x = m, h, n
 * with the three shapes of rate function of the 1952 paper, each {A, V_half, k}, u = (V - V_half)/k:
 *     exponential  A exp(-u)                 beta_m, alpha_h, beta_n
 *     sigmoid      A / (1 + exp(-u))         beta_h
 *     linoid       A k u / (1 - exp(-u))     alpha_m, alpha_n  (-> A k at u = 0; the series 1 + u/2 + u^2/12 is used for
 *                                            |u| < 0.05, where it is exact to 1e-8 and the quotient loses digits)
 * Rate index f: 0 alpha_m, 1 beta_m, 2 alpha_h, 3 beta_h, 4 alpha_n, 5 beta_n.
 * ---------------------------------------------------------------------------------------- */
enum { ORC_HH_EXP = 0, ORC_HH_SIGMOID = 1, ORC_HH_LINOID = 2 };

int orc_hh_kind(int f)
{
    return (f == 0 || f == 4) ? ORC_HH_LINOID : (f == 3 ? ORC_HH_SIGMOID : ORC_HH_EXP);
}

/* The definition, in double with libm's exp. */
double orc_hh_rate(int f, double A, double v_half, double k, double V)
{
    const double u = (V - v_half) * (1.0 / k);
    switch (orc_hh_kind(f)) {
    case ORC_HH_LINOID:
        if (fabs(u) < 0.05) return (A * k) * fma(u, fma(u, 1.0 / 12.0, 0.5), 1.0);
        return (A * k) * (u / (1.0 - exp(-u)));
    case ORC_HH_SIGMOID: return A / (1.0 + exp(-u));
    default: return A * exp(-u);
    }
}

/* exp for the fp32-faithful mode: every step one correctly rounded binary32 operation, so that the CUDA kernels can
 * follow it bit for bit (Hodgkin-Huxley).  Argument clamped to [-87, 88] (a rate
 * function never needs more); n = rint(x log2 e); r = x - n ln 2 in two steps (Cody-Waite); degree-7 Taylor polynomial
 * of e^r on |r| <= ln2 / 2 (remainder 5e-9) by Horner with fmaf; scaled by 2^n through the exponent field. */
float orc_exp32(float x)
{
    if (x > 88.0f) x = 88.0f;
    if (x < -87.0f) x = -87.0f;
    const float n = rintf(x * 0x1.715476p+0f);
    float r = fmaf(n, -0x1.62e400p-1f, x);
    r = fmaf(n, -0x1.7f7d1cp-20f, r);
    float p = 0x1.a01a02p-13f;                 /* 1/5040 */
    p = fmaf(p, r, 0x1.6c16c2p-10f);           /* 1/720  */
    p = fmaf(p, r, 0x1.111112p-7f);            /* 1/120  */
    p = fmaf(p, r, 0x1.555556p-5f);            /* 1/24   */
    p = fmaf(p, r, 0x1.555556p-3f);            /* 1/6    */
    p = fmaf(p, r, 0.5f);
    p = fmaf(p, r, 1.0f);
    p = fmaf(p, r, 1.0f);
    union { uint32_t u; float f; } s;
    s.u = (uint32_t)((int32_t)n + 127) << 23;  /* 2^n, n in [-126, 127] */
    return p * s.f;
}

/* One rate in the fp32-faithful order: ak = (float)(A) or (float)(A k), inv_k = (float)(1/k). */
float orc_hh_rate32(int f, float ak, float v_half, float inv_k, float V)
{
    const float u = (V - v_half) * inv_k;
    switch (orc_hh_kind(f)) {
    case ORC_HH_LINOID:
        if (fabsf(u) < 0.05f) return ak * fmaf(u, fmaf(u, 0x1.555556p-4f, 0.5f), 1.0f);
        return ak * (u / (1.0f - orc_exp32(-u)));
    case ORC_HH_SIGMOID: return ak / (1.0f + orc_exp32(-u));
    default: return ak * orc_exp32(-u);
    }
}

/* ------------------------------------------------------------------------------------------
 * The simulator
 * ---------------------------------------------------------------------------------------- */
enum { ORC_CLASS_FLOATS = 40 };

typedef struct {
    /* as given (fp32 at the boundary) */
    float a, b, c_reset, d, k2, k1, k0, v_peak, tau_syn_ms, refractory_ms, drive_rate_hz, drive_kick, psc_alpha;
    /* Hodgkin-Huxley class (model == 1): capacitance, conductances, reversal potentials, resting potential, and
     * {A, V_half, k} of the six rate functions alpha_m, beta_m, alpha_h, beta_h, alpha_n, beta_n */
    float model, hh_c, hh_g_na, hh_g_k, hh_g_l, hh_e_na, hh_e_k, hh_e_l, hh_v_rest, hh_rate[6][3];
    int hh;              /* model == 1 */
    double hh_dt_c, hh_ak[6], hh_inv_k[6];      /* dt/C, A (A*k for the two linoid rates), 1/k: formed once in double */
    float hh_dt_c_f, hh_ak_f[6], hh_inv_k_f[6]; /* ... and rounded once for the fp32-faithful mode */
    /* derived */
    int direct;          /* tau_syn_ms <= 0: arriving weight jumps V itself */
    int alpha;           /* psc_alpha != 0: alpha-function PSC (eq. 27, 29, 30) instead of the exponential one (eq. 26) */
    double keep_s;       /* 1 - dt/tau_s */
    float keep_s_f;
    double a2, two_a;    /* alpha-function: a^2 and 2a with a = 1/tau_s (per ms) */
    float a2_f, two_a_f;
    uint32_t R;          /* refractory steps */
    uint32_t drive_thr;
    int64_t kick_fx;
} orc_class;

typedef struct orc_net {
    uint32_t n, dim, D, n_classes, mode, obs_stride;
    uint64_t E, seed;
    float dt_f;
    double dt;
    orc_class *cls_tab;
    uint64_t *row;      /* [n+1] CSR by source */
    uint32_t *tgt;      /* [E] */
    int64_t *w_fx;      /* [E] */
    uint32_t *delay;    /* [E] steps */
    uint8_t *cls;       /* [n] */
    float *bias;        /* [n] or NULL */
    /* state; mode 0 uses the double arrays, mode 1 the float arrays */
    double *V, *W, *r, *p, *c, *acc, *hm, *hh;    /* hm, hh: the gates m and h of Hodgkin-Huxley vertices (n lives in W) */
    float *Vf, *Wf, *rf, *pf, *cf, *accf, *hmf, *hhf;
    uint32_t *refr;
    int64_t *ring;      /* [D][n] */
    int64_t *consumed;  /* [n] I_fx (kick included) consumed by the last step */
    uint8_t *fired;     /* [n] scratch */
    /* observation parameters */
    double keep_c, ca_jump, obs_gain, obs_offset, obs_sigma;
    float keep_c_f, ca_jump_f;
    /* history */
    uint64_t t;
    uint32_t words;     /* ceil(n/32) */
    uint32_t *raster;   /* [t][words], grows */
    uint64_t raster_cap;
    double *trace;      /* [frames][n], grows */
    uint64_t frames, trace_cap;
    /* counters */
    uint64_t spikes, delivered, kicks;
    int64_t mass_delivered, mass_consumed; /* fixed-point sums, kicks excluded */
    int overflow;       /* a ring slot left the int32 range */
    /* plastic weights (orc_enable_stdp; PAPER.md:323-349 eq. 32-33, :103-119 eq. 9): every weight a state of its own */
    int plastic;
    double stdp_alpha, stdp_beta;   /* as given (fp32 at the boundary), in double */
    float stdp_dta_f, stdp_beta_f;  /* (float)(dt alpha) rounded once, beta: the fp32-faithful mode's constants */
    double *wd;         /* [E] w_ij(t), mode 0 */
    float *wf;          /* [E] w_ij(t), mode 1 */
    int64_t *age;       /* [D+1][n] row tau mod (D+1): s_j(tau) of eq. 32 in steps, -1 = j has not fired yet (reading #23) */
    int64_t *I_in;      /* [n] eq. 30's sum at the step in hand, fixed point */
} orc_net;

void orc_destroy(orc_net *o)
{
    if (!o) return;
    free(o->cls_tab); free(o->row); free(o->tgt); free(o->w_fx); free(o->delay); free(o->cls);
    free(o->bias); free(o->V); free(o->W); free(o->r); free(o->c); free(o->acc);
    free(o->Vf); free(o->Wf); free(o->rf); free(o->pf); free(o->cf); free(o->accf); free(o->p);
    free(o->hm); free(o->hh); free(o->hmf); free(o->hhf);
    free(o->refr); free(o->ring); free(o->consumed); free(o->fired); free(o->raster); free(o->trace);
    free(o->wd); free(o->wf); free(o->age); free(o->I_in);
    free(o);
}

/*
 * class_params: [n_classes][ORC_CLASS_FLOATS = 40] floats in the order
 *   a, b, c_reset, d, k2, k1, k0, v_peak, tau_syn_ms, refractory_ms, drive_rate_hz, drive_kick, psc_alpha,
 *   model, hh_c, hh_g_na, hh_g_k, hh_g_l, hh_e_na, hh_e_k, hh_e_l, hh_v_rest, then {A, V_half, k} of alpha_m, beta_m,
 *   alpha_h, beta_h, alpha_n, beta_n.
 * delays: [E] steps, or NULL => eq. 25 from positions and speed.
 * Returns NULL on a malformed graph (row offsets, target range, delay outside [1, D-1]).
 * Initial state (reading #15): V = -70, W = b*V, r = c = 0, refr = 0, ring zero.
 */
orc_net *orc_create(uint32_t n, uint32_t dim, uint64_t E, uint32_t D, float dt_ms, float speed,
                    uint32_t n_classes, const float *class_params, const float *positions,
                    const uint64_t *row_offsets, const uint32_t *targets, const float *weights,
                    const uint8_t *delays, const uint8_t *vertex_class, const float *bias,
                    float tau_ca_ms, float ca_jump, float obs_gain, float obs_offset,
                    float obs_sigma, uint32_t obs_stride, uint64_t seed, uint32_t mode)
{
    if (D < 2 || n_classes < 1 || mode > 1) return NULL;
    orc_net *o = (orc_net *)calloc(1, sizeof(orc_net));
    if (!o) return NULL;
    o->n = n; o->dim = dim; o->E = E; o->D = D; o->n_classes = n_classes; o->mode = mode;
    o->obs_stride = obs_stride; o->seed = seed; o->dt_f = dt_ms; o->dt = (double)dt_ms;
    o->words = (n + 31) / 32;
    size_t n1 = n ? n : 1, e1 = E ? E : 1;
    o->cls_tab = (orc_class *)calloc(n_classes, sizeof(orc_class));
    o->row = (uint64_t *)malloc((n1 + 1) * sizeof(uint64_t));
    o->tgt = (uint32_t *)malloc(e1 * sizeof(uint32_t));
    o->w_fx = (int64_t *)malloc(e1 * sizeof(int64_t));
    o->delay = (uint32_t *)malloc(e1 * sizeof(uint32_t));
    o->cls = (uint8_t *)malloc(n1);
    o->refr = (uint32_t *)calloc(n1, sizeof(uint32_t));
    o->ring = (int64_t *)calloc((size_t)D * n1, sizeof(int64_t));
    o->consumed = (int64_t *)calloc(n1, sizeof(int64_t));
    o->fired = (uint8_t *)calloc(n1, 1);
    o->V = (double *)calloc(n1, sizeof(double)); o->W = (double *)calloc(n1, sizeof(double));
    o->r = (double *)calloc(n1, sizeof(double)); o->c = (double *)calloc(n1, sizeof(double));
    o->acc = (double *)calloc(n1, sizeof(double));
    o->p = (double *)calloc(n1, sizeof(double)); o->pf = (float *)calloc(n1, sizeof(float));
    o->Vf = (float *)calloc(n1, sizeof(float)); o->Wf = (float *)calloc(n1, sizeof(float));
    o->rf = (float *)calloc(n1, sizeof(float)); o->cf = (float *)calloc(n1, sizeof(float));
    o->accf = (float *)calloc(n1, sizeof(float));
    o->hm = (double *)calloc(n1, sizeof(double)); o->hh = (double *)calloc(n1, sizeof(double));
    o->hmf = (float *)calloc(n1, sizeof(float)); o->hhf = (float *)calloc(n1, sizeof(float));
    if (bias) {
        o->bias = (float *)malloc(n1 * sizeof(float));
        memcpy(o->bias, bias, (size_t)n * sizeof(float));
    }
    for (uint32_t k = 0; k < n_classes; ++k) {
        const float *p = class_params + ORC_CLASS_FLOATS * k;
        orc_class *q = &o->cls_tab[k];
        q->a = p[0]; q->b = p[1]; q->c_reset = p[2]; q->d = p[3];
        q->k2 = p[4]; q->k1 = p[5]; q->k0 = p[6]; q->v_peak = p[7];
        q->tau_syn_ms = p[8]; q->refractory_ms = p[9]; q->drive_rate_hz = p[10]; q->drive_kick = p[11];
        q->psc_alpha = p[12];
        q->model = p[13]; q->hh = q->model == 1.0f;
        q->hh_c = p[14]; q->hh_g_na = p[15]; q->hh_g_k = p[16]; q->hh_g_l = p[17];
        q->hh_e_na = p[18]; q->hh_e_k = p[19]; q->hh_e_l = p[20]; q->hh_v_rest = p[21];
        for (int f = 0; f < 6; ++f)
            for (int i = 0; i < 3; ++i) q->hh_rate[f][i] = p[22 + 3 * f + i];
        if (q->hh) {
            q->hh_dt_c = (double)dt_ms / (double)q->hh_c;
            q->hh_dt_c_f = (float)q->hh_dt_c;
            for (int f = 0; f < 6; ++f) {
                const double A = q->hh_rate[f][0], kk = q->hh_rate[f][2];
                q->hh_ak[f] = orc_hh_kind(f) == ORC_HH_LINOID ? A * kk : A;
                q->hh_inv_k[f] = 1.0 / kk;
                q->hh_ak_f[f] = (float)q->hh_ak[f];
                q->hh_inv_k_f[f] = (float)q->hh_inv_k[f];
            }
        }
        q->direct = !(q->tau_syn_ms > 0.0f);
        q->alpha = !q->direct && q->psc_alpha != 0.0f;
        q->keep_s = q->direct ? 0.0 : orc_keep(dt_ms, q->tau_syn_ms);
        q->keep_s_f = (float)q->keep_s;
        if (q->alpha) {      /* a = 1/tau_s: constants formed once in double, rounded once for the fp32-faithful mode */
            q->a2 = 1.0 / ((double)q->tau_syn_ms * (double)q->tau_syn_ms);
            q->two_a = 2.0 / (double)q->tau_syn_ms;
            q->a2_f = (float)q->a2;
            q->two_a_f = (float)q->two_a;
        }
        q->R = orc_refractory_steps(q->refractory_ms, dt_ms);
        q->drive_thr = orc_drive_threshold(q->drive_rate_hz, dt_ms);
        q->kick_fx = orc_quantise(q->drive_kick);
    }
    o->keep_c = tau_ca_ms > 0.0f ? orc_keep(dt_ms, tau_ca_ms) : 0.0;
    o->keep_c_f = (float)o->keep_c;
    o->ca_jump = (double)ca_jump; o->ca_jump_f = ca_jump;
    o->obs_gain = obs_gain; o->obs_offset = obs_offset; o->obs_sigma = obs_sigma;

    int bad = 0;
    memcpy(o->row, row_offsets, ((size_t)n + 1) * sizeof(uint64_t));
    if (o->row[0] != 0 || o->row[n] != E) bad = 1;
    for (uint32_t i = 0; i < n && !bad; ++i)
        if (o->row[i + 1] < o->row[i]) bad = 1;
    for (uint32_t i = 0; i < n && !bad; ++i) {
        if (vertex_class[i] >= n_classes) { bad = 1; break; }
        o->cls[i] = vertex_class[i];
        for (uint64_t e = o->row[i]; e < o->row[i + 1]; ++e) {
            uint32_t m = targets[e];
            if (m >= n) { bad = 1; break; }
            o->tgt[e] = m;
            o->w_fx[e] = orc_quantise(weights[e]);
            o->delay[e] = delays ? (uint32_t)delays[e]
                                 : orc_delay_steps(positions + (size_t)i * dim, positions + (size_t)m * dim,
                                                   dim, speed, dt_ms);
            if (o->delay[e] < 1 || o->delay[e] > D - 1) { bad = 1; break; }
        }
    }
    if (bad) { orc_destroy(o); return NULL; }
    for (uint32_t j = 0; j < n; ++j) {
        const orc_class *q = &o->cls_tab[o->cls[j]];
        if (q->hh) {         /* at rest: V = hh_v_rest, every gate at its steady state alpha / (alpha + beta) for that V */
            double g[3];
            for (int x = 0; x < 3; ++x) {
                const double al = orc_hh_rate(2 * x, q->hh_rate[2 * x][0], q->hh_rate[2 * x][1], q->hh_rate[2 * x][2], q->hh_v_rest);
                const double be = orc_hh_rate(2 * x + 1, q->hh_rate[2 * x + 1][0], q->hh_rate[2 * x + 1][1], q->hh_rate[2 * x + 1][2], q->hh_v_rest);
                g[x] = al / (al + be);
            }
            o->V[j] = q->hh_v_rest; o->hm[j] = g[0]; o->hh[j] = g[1]; o->W[j] = g[2];
            o->Vf[j] = q->hh_v_rest; o->hmf[j] = (float)g[0]; o->hhf[j] = (float)g[1]; o->Wf[j] = (float)g[2];
            continue;
        }
        o->V[j] = -70.0; o->W[j] = (double)q->b * -70.0;
        o->Vf[j] = -70.0f; o->Wf[j] = q->b * -70.0f;
    }
    return o;
}

static int orc_reserve_history(orc_net *o, uint64_t n_steps)
{
    if (o->t + n_steps > o->raster_cap) {
        uint64_t cap = o->raster_cap ? o->raster_cap : 64;
        while (cap < o->t + n_steps) cap *= 2;
        uint32_t *p = (uint32_t *)realloc(o->raster, (size_t)cap * (o->words ? o->words : 1) * sizeof(uint32_t));
        if (!p) return -1;
        o->raster = p; o->raster_cap = cap;
    }
    if (o->obs_stride) {
        uint64_t need = (o->t + n_steps) / o->obs_stride;
        if (need > o->trace_cap) {
            uint64_t cap = o->trace_cap ? o->trace_cap : 16;
            while (cap < need) cap *= 2;
            double *p = (double *)realloc(o->trace, (size_t)cap * (o->n ? o->n : 1) * sizeof(double));
            if (!p) return -1;
            o->trace = p; o->trace_cap = cap;
        }
    }
    return 0;
}

/* Steps 1-5 and 7 for vertex j in double.  Returns fired. */
static int orc_vertex_fp64(orc_net *o, uint32_t j, int64_t I_fx)
{
    const orc_class *q = &o->cls_tab[o->cls[j]];
    const double dt = o->dt;
    const double a = q->a, b = q->b, k2 = q->k2, k1 = q->k1, k0 = q->k0;
    double V = o->V[j], W = o->W[j], r = o->r[j];
    double I = (double)I_fx * (1.0 / 65536.0);
    double U = o->bias ? (double)o->bias[j] : 0.0;                         /* U_j(t), eq. 28 */
    int fired = (o->refr[j] == 0) && (V >= (double)q->v_peak);            /* eq. 31 */
    double W_euler = fma(dt, a * fma(b, V, -W), W);                        /* eq. 24, W line */
    double Vn, Wn;
    if (fired) {                                                           /* eq. 24 "otherwise" */
        Vn = q->c_reset; Wn = W + (double)q->d; o->refr[j] = q->R;
    } else if (o->refr[j] > 0) {                                           /* refractory hold */
        Vn = q->c_reset; Wn = W_euler; o->refr[j] -= 1;
    } else {                                                               /* eq. 28, V < V_peak */
        double t1 = fma(k2, V, k1);
        double t2 = fma(t1, V, k0);
        double t3 = t2 - W;
        double t4 = q->direct ? t3 : t3 + r;
        if (o->bias) t4 = t4 + U;
        Vn = fma(dt, t4, V);
        if (q->direct) Vn = Vn + I;
        Wn = W_euler;
    }
    o->V[j] = Vn; o->W[j] = Wn;
    if (q->alpha) {                                                        /* eq. 29-30 (impulse reading #4: p jumps by I) */
        double pp = o->p[j];
        double q2 = fma(q->two_a, pp, q->a2 * r);
        o->r[j] = fma(dt, pp, r);                                          /* H_r = r + dt p */
        o->p[j] = fma(-dt, q2, pp) + I;                                    /* H_p = p + dt(-a^2 r - 2a p) + arrivals */
    } else if (!q->direct) {
        o->r[j] = fma(q->keep_s, r, I);                                    /* eq. 26 */
    }
    if (o->obs_stride) {
        double cn = fma(o->keep_c, o->c[j], fired ? o->ca_jump : 0.0);     /* H_c */
        o->c[j] = cn;
        o->acc[j] = o->acc[j] + cn;
    }
    return fired;
}

/* The same sequence, every operation one correctly rounded binary32 operation. */
static int orc_vertex_fp32(orc_net *o, uint32_t j, int64_t I_fx)
{
    const orc_class *q = &o->cls_tab[o->cls[j]];
    const float dt = o->dt_f;
    float V = o->Vf[j], W = o->Wf[j], r = o->rf[j];
    float If = (float)(int32_t)I_fx * 0x1p-16f;
    float U = o->bias ? o->bias[j] : 0.0f;
    int fired = (o->refr[j] == 0) && (V >= q->v_peak);
    float u1 = fmaf(q->b, V, -W);
    float u2 = q->a * u1;
    float W_euler = fmaf(dt, u2, W);
    float Vn, Wn;
    if (fired) {
        Vn = q->c_reset; Wn = W + q->d; o->refr[j] = q->R;
    } else if (o->refr[j] > 0) {
        Vn = q->c_reset; Wn = W_euler; o->refr[j] -= 1;
    } else {
        float t1 = fmaf(q->k2, V, q->k1);
        float t2 = fmaf(t1, V, q->k0);
        float t3 = t2 - W;
        float t4 = q->direct ? t3 : t3 + r;
        if (o->bias) t4 = t4 + U;
        Vn = fmaf(dt, t4, V);
        if (q->direct) Vn = Vn + If;
        Wn = W_euler;
    }
    o->Vf[j] = Vn; o->Wf[j] = Wn;
    if (q->alpha) {
        float pp = o->pf[j];
        float q1 = q->a2_f * r;
        float q2 = fmaf(q->two_a_f, pp, q1);
        float p1 = fmaf(-dt, q2, pp);
        o->rf[j] = fmaf(dt, pp, r);
        o->pf[j] = p1 + If;
    } else if (!q->direct) {
        o->rf[j] = fmaf(q->keep_s_f, r, If);
    }
    if (o->obs_stride) {
        float cn = fmaf(o->keep_c_f, o->cf[j], fired ? o->ca_jump_f : 0.0f);
        o->cf[j] = cn;
        o->accf[j] = o->accf[j] + cn;
    }
    return fired;
}

/* Steps 2-5 for a Hodgkin-Huxley vertex in double: detect on the state at t (eq. 31), forward Euler (eq. 19) of the four
 * textbook equations from the state at t, the PSC and the calcium as for every class.  There is no reset: `refr` only
 * keeps one action potential (V stays above v_peak for many steps) from being detected again for refractory_ms. */
static int orc_vertex_hh_fp64(orc_net *o, uint32_t j, int64_t I_fx)
{
    const orc_class *q = &o->cls_tab[o->cls[j]];
    const double V = o->V[j], m = o->hm[j], h = o->hh[j], n = o->W[j], r = o->r[j];
    const double I = (double)I_fx * (1.0 / 65536.0);
    int fired = (o->refr[j] == 0) && (V >= (double)q->v_peak);
    if (fired) o->refr[j] = q->R;
    else if (o->refr[j] > 0) o->refr[j] -= 1;
    double rate[6];
    for (int f = 0; f < 6; ++f) rate[f] = orc_hh_rate(f, q->hh_rate[f][0], q->hh_rate[f][1], q->hh_rate[f][2], V);
    const double i_na = (((double)q->hh_g_na * ((m * m) * m)) * h) * (V - (double)q->hh_e_na);
    const double i_k = ((double)q->hh_g_k * ((n * n) * (n * n))) * (V - (double)q->hh_e_k);
    const double i_l = (double)q->hh_g_l * (V - (double)q->hh_e_l);
    double s = r - ((i_na + i_k) + i_l);
    if (o->bias) s = s + (double)o->bias[j];
    o->V[j] = fma(q->hh_dt_c, s, V);
    if (q->direct) o->V[j] = o->V[j] + I;      /* DESIGN.md reading #4: tau_syn_ms <= 0, the arriving weight jumps V itself */
    o->hm[j] = fma(o->dt, fma(-rate[1], m, rate[0] * (1.0 - m)), m);
    o->hh[j] = fma(o->dt, fma(-rate[3], h, rate[2] * (1.0 - h)), h);
    o->W[j] = fma(o->dt, fma(-rate[5], n, rate[4] * (1.0 - n)), n);
    if (q->alpha) {
        double pp = o->p[j];
        double q2 = fma(q->two_a, pp, q->a2 * r);
        o->r[j] = fma(o->dt, pp, r);
        o->p[j] = fma(-o->dt, q2, pp) + I;
    } else if (!q->direct) {
        o->r[j] = fma(q->keep_s, r, I);
    }
    if (o->obs_stride) {
        double cn = fma(o->keep_c, o->c[j], fired ? o->ca_jump : 0.0);
        o->c[j] = cn;
        o->acc[j] = o->acc[j] + cn;
    }
    return fired;
}

/* The same sequence, every operation one correctly rounded binary32 operation (exp by orc_exp32). */
static int orc_vertex_hh_fp32(orc_net *o, uint32_t j, int64_t I_fx)
{
    const orc_class *q = &o->cls_tab[o->cls[j]];
    const float dt = o->dt_f;
    const float V = o->Vf[j], m = o->hmf[j], h = o->hhf[j], n = o->Wf[j], r = o->rf[j];
    const float If = (float)(int32_t)I_fx * 0x1p-16f;
    int fired = (o->refr[j] == 0) && (V >= q->v_peak);
    if (fired) o->refr[j] = q->R;
    else if (o->refr[j] > 0) o->refr[j] -= 1;
    float rate[6];
    for (int f = 0; f < 6; ++f) rate[f] = orc_hh_rate32(f, q->hh_ak_f[f], q->hh_rate[f][1], q->hh_inv_k_f[f], V);
    const float m2 = m * m, m3 = m2 * m, gna = (q->hh_g_na * m3) * h, i_na = gna * (V - q->hh_e_na);
    const float n2 = n * n, n4 = n2 * n2, i_k = (q->hh_g_k * n4) * (V - q->hh_e_k);
    const float i_l = q->hh_g_l * (V - q->hh_e_l);
    float s = r - ((i_na + i_k) + i_l);
    if (o->bias) s = s + o->bias[j];
    o->Vf[j] = fmaf(q->hh_dt_c_f, s, V);
    if (q->direct) o->Vf[j] = o->Vf[j] + If;   /* reading #4, as above */
    o->hmf[j] = fmaf(dt, fmaf(-rate[1], m, rate[0] * (1.0f - m)), m);
    o->hhf[j] = fmaf(dt, fmaf(-rate[3], h, rate[2] * (1.0f - h)), h);
    o->Wf[j] = fmaf(dt, fmaf(-rate[5], n, rate[4] * (1.0f - n)), n);
    if (q->alpha) {
        float pp = o->pf[j];
        float q1 = q->a2_f * r;
        float q2 = fmaf(q->two_a_f, pp, q1);
        float p1 = fmaf(-dt, q2, pp);
        o->rf[j] = fmaf(dt, pp, r);
        o->pf[j] = p1 + If;
    } else if (!q->direct) {
        o->rf[j] = fmaf(q->keep_s_f, r, If);
    }
    if (o->obs_stride) {
        float cn = fmaf(o->keep_c_f, o->cf[j], fired ? o->ca_jump_f : 0.0f);
        o->cf[j] = cn;
        o->accf[j] = o->accf[j] + cn;
    }
    return fired;
}

/* ---- plastic weights: PAPER.md:323-349 (section 3.2.3, eq. 32-33) on top of eq. 30 (:311) and eq. 9 (:103-119) -------------
 * Written for sizes the pure-Python definition (oracle/stdp_definition.py) cannot reach; pinned against it and against eq. 33's
 * closed form in tests/test_oracle_stdp.py.  Nothing is pushed into a ring here: eq. 30 weighs the spike of k arriving at j at
 * step t with w_kj(t), the weight AT THE ARRIVAL step, so the sum is PULLED at step t from the raster history by visiting every
 * edge, and eq. 33 is then applied to every edge, one by one, in the paper's order:
 *   s_j(t + dt) = (1 - spd(V_j(t))) (s_j(t) + dt)                                                      eq. 32, kept in steps
 *   q_ij(t) = (s~_i(t - tau_ij) - s~_j(t)) max(spd(V_i(t - tau_ij)), spd(V_j(t)))                       eq. 33
 *   w_ij(t + dt) = w_ij(t) + dt alpha sign(q_ij) exp(-beta |q_ij|)
 * with s~ the age after eq. 32's reset factor (reading #22: 0 for a vertex spiking at the step) and no age before the first
 * spike (reading #23).  Hence, per edge i -> j of delay d at step t (pre: i fired at t - d; post: j fires at t):
 *   pre and not post:  q = -s_j(t)        the weight falls by dt alpha exp(-beta s_j(t))       if s_j(t) > 0
 *   post and not pre:  q = +s_i(t - d)    the weight rises by dt alpha exp(-beta s_i(t - d))   if s_i(t - d) > 0
 *   both, neither, or an age of 0 (sign(0) = 0):  no change.
 * mode 0: weights, ages and the exponential in double (libm).  mode 1 (fp32-faithful): one
 * rounded binary32 operation each, age = (float)steps * dt, dw = (float)(dt alpha) * exp32(-(beta * age)), w -+ dw.
 * Either way an arriving weight enters eq. 30's fixed-point sum as rint(w 2^16), ties to even (mode 1 saturates at int32 as
 * the conversion instruction does), like every static weight. */
int orc_enable_stdp(orc_net *o, float alpha, float beta)
{
    if (!o || o->t != 0 || !(beta >= 0.0f)) return -1;
    o->plastic = 1;
    o->stdp_alpha = (double)alpha; o->stdp_beta = (double)beta;
    o->stdp_dta_f = (float)(o->dt * (double)alpha); o->stdp_beta_f = beta;
    const size_t E1 = o->E ? (size_t)o->E : 1, n1 = o->n ? o->n : 1;
    o->wd = (double *)malloc(E1 * sizeof(double));
    o->wf = (float *)malloc(E1 * sizeof(float));
    o->age = (int64_t *)malloc((size_t)(o->D + 1) * n1 * sizeof(int64_t));
    o->I_in = (int64_t *)calloc(n1, sizeof(int64_t));
    if (!o->wd || !o->wf || !o->age || !o->I_in) return -1;
    for (uint64_t e = 0; e < o->E; ++e) {          /* the weights start at the quantised values the static network has */
        o->wd[e] = (double)o->w_fx[e] / 65536.0;
        o->wf[e] = (float)o->wd[e];
    }
    for (size_t k = 0; k < (size_t)(o->D + 1) * n1; ++k) o->age[k] = -1;
    return 0;
}

static inline int orc_fired_at(const orc_net *o, uint64_t t, uint32_t i)
{
    return (o->raster[(size_t)t * o->words + (i >> 5)] >> (i & 31)) & 1u;
}

static int orc_step_plastic(orc_net *o, uint64_t n_steps)
{
    const uint32_t n = o->n, D = o->D;
    for (uint64_t s = 0; s < n_steps; ++s) {
        const uint64_t t = o->t;
        uint32_t *rast = o->raster + (size_t)t * o->words;
        memset(rast, 0, (size_t)o->words * sizeof(uint32_t));
        memset(o->I_in, 0, (size_t)n * sizeof(int64_t));
        /* eq. 30 at step t: every edge whose source fired exactly `delay` steps ago contributes its CURRENT weight */
        uint64_t delivered = 0;
        int64_t mass_delivered = 0;
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : delivered, mass_delivered)
        for (int64_t ii = 0; ii < (int64_t)n; ++ii) {
            for (uint64_t e = o->row[ii]; e < o->row[ii + 1]; ++e) {
                const uint64_t d = o->delay[e];
                if (t < d || !orc_fired_at(o, t - d, (uint32_t)ii)) continue;
                int64_t w_fx;
                if (o->mode) {
                    const float sc = o->wf[e] * 65536.0f;
                    w_fx = sc != sc ? 0 : sc >= 2147483648.0f ? 2147483647ll : sc <= -2147483648.0f ? -2147483648ll : (int64_t)rintf(sc);
                } else {
                    w_fx = (int64_t)llrint(o->wd[e] * 65536.0);
                }
#pragma omp atomic
                o->I_in[o->tgt[e]] += w_fx;
                delivered += 1;
                mass_delivered += w_fx;
            }
        }
        uint64_t spikes = 0, kicks = 0;
        int64_t mass_consumed = 0;
        int overflow = 0;
#pragma omp parallel for schedule(static) reduction(+ : spikes, kicks, mass_consumed) reduction(| : overflow)
        for (int64_t jj = 0; jj < (int64_t)n; ++jj) {      /* the vertex transition, exactly as in orc_step */
            const uint32_t j = (uint32_t)jj;
            int64_t I_fx = o->I_in[j];
            if (I_fx > 2147483647ll || I_fx < -2147483648ll) overflow = 1;
            mass_consumed += I_fx;
            const orc_class *q = &o->cls_tab[o->cls[j]];
            if (q->drive_thr && orc_word(o->seed, ORC_STREAM_DRIVE, j, t) < q->drive_thr) {
                I_fx += q->kick_fx;
                kicks += 1;
            }
            o->consumed[j] = I_fx;
            int f = q->hh ? (o->mode ? orc_vertex_hh_fp32(o, j, I_fx) : orc_vertex_hh_fp64(o, j, I_fx))
                          : (o->mode ? orc_vertex_fp32(o, j, I_fx) : orc_vertex_fp64(o, j, I_fx));
            o->fired[j] = (uint8_t)f;
            spikes += (uint64_t)f;
        }
        for (uint32_t j = 0; j < n; ++j)
            if (o->fired[j]) rast[j >> 5] |= 1u << (j & 31);
        /* eq. 33, edge by edge */
        const int64_t *age_t = o->age + (size_t)(t % (D + 1)) * n;
#pragma omp parallel for schedule(dynamic, 64)
        for (int64_t ii = 0; ii < (int64_t)n; ++ii) {
            for (uint64_t e = o->row[ii]; e < o->row[ii + 1]; ++e) {
                const uint64_t d = o->delay[e];
                const uint32_t j = o->tgt[e];
                const int pre = t >= d && orc_fired_at(o, t - d, (uint32_t)ii);
                const int post = o->fired[j];
                if (pre == post) continue;                                  /* neither: max(..) = 0; both: q = 0 */
                int64_t steps;
                if (pre) steps = age_t[j];                                  /* q = -s_j(t) */
                else if (t >= d) steps = o->age[(size_t)((t - d) % (D + 1)) * n + (uint32_t)ii];   /* q = +s_i(t - d) */
                else steps = -1;                                            /* i has no age d steps before the start */
                if (steps <= 0) continue;                                   /* no age yet (reading #23), or q = 0 */
                if (o->mode) {
                    const float a = (float)steps * o->dt_f;
                    const float dw = o->stdp_dta_f * orc_exp32(-(o->stdp_beta_f * a));
                    o->wf[e] = pre ? o->wf[e] - dw : o->wf[e] + dw;
                } else {
                    const double a = (double)steps * o->dt;
                    const double dw = (o->dt * o->stdp_alpha) * exp(-(o->stdp_beta * a));
                    o->wd[e] = pre ? o->wd[e] - dw : o->wd[e] + dw;
                }
            }
        }
        /* eq. 32: s_j(t + dt) = (1 - spd(V_j(t))) (s_j(t) + dt), in steps; no age before the first spike */
        int64_t *age_n = o->age + (size_t)((t + 1) % (D + 1)) * n;
        for (uint32_t j = 0; j < n; ++j) age_n[j] = o->fired[j] ? 0 : (age_t[j] < 0 ? -1 : age_t[j] + 1);
        if (o->obs_stride && (t + 1) % o->obs_stride == 0) {   /* step 7: emit one frame (as in orc_step) */
            const uint64_t frame = (t + 1) / o->obs_stride - 1;
            double *z = o->trace + (size_t)frame * n;
            for (uint32_t j = 0; j < n; ++j) {
                double sum = o->mode ? (double)o->accf[j] : o->acc[j];
                double g = o->obs_sigma != 0.0 ? orc_gauss(o->seed, j, frame) : 0.0;
                z[j] = o->obs_gain * (sum / (double)o->obs_stride) + o->obs_offset + o->obs_sigma * g;
                o->acc[j] = 0.0; o->accf[j] = 0.0f;
            }
            o->frames = frame + 1;
        }
        o->spikes += spikes; o->kicks += kicks; o->delivered += delivered;
        o->mass_consumed += mass_consumed; o->mass_delivered += mass_delivered;
        o->overflow |= overflow;
        o->t = t + 1;
    }
    return o->overflow ? -2 : 0;
}

/* w_ij(t) of every edge, in the caller's (CSR) edge order; the static weights when orc_enable_stdp was not called. */
void orc_get_weights(const orc_net *o, double *out)
{
    for (uint64_t e = 0; e < o->E; ++e)
        out[e] = !o->plastic ? (double)o->w_fx[e] / 65536.0 : o->mode ? (double)o->wf[e] : o->wd[e];
}

/* Advance n_steps.  Returns 0, -1 (out of memory) or -2 (a ring slot left the int32 range). */
int orc_step(orc_net *o, uint64_t n_steps, int n_threads)
{
    if (orc_reserve_history(o, n_steps)) return -1;
    if (o->plastic) {
#ifdef _OPENMP
        if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
        return orc_step_plastic(o, n_steps);
    }
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#else
    (void)n_threads;
#endif
    const uint32_t n = o->n, D = o->D;
    for (uint64_t s = 0; s < n_steps; ++s) {
        const uint64_t t = o->t;
        int64_t *slot = o->ring + (size_t)(t % D) * n;
        uint32_t *rast = o->raster + (size_t)t * o->words;
        memset(rast, 0, (size_t)o->words * sizeof(uint32_t));
        uint64_t spikes = 0, kicks = 0;
        int64_t mass_consumed = 0;
        int overflow = 0;
#pragma omp parallel for schedule(static) reduction(+ : spikes, kicks, mass_consumed) reduction(| : overflow)
        for (int64_t jj = 0; jj < (int64_t)n; ++jj) {
            const uint32_t j = (uint32_t)jj;
            int64_t I_fx = slot[j];                         /* step 1: read and clear */
            slot[j] = 0;
            if (I_fx > 2147483647ll || I_fx < -2147483648ll) overflow = 1;
            mass_consumed += I_fx;
            const orc_class *q = &o->cls_tab[o->cls[j]];
            if (q->drive_thr && orc_word(o->seed, ORC_STREAM_DRIVE, j, t) < q->drive_thr) {
                I_fx += q->kick_fx;
                kicks += 1;
            }
            o->consumed[j] = I_fx;
            int f = q->hh ? (o->mode ? orc_vertex_hh_fp32(o, j, I_fx) : orc_vertex_hh_fp64(o, j, I_fx))
                          : (o->mode ? orc_vertex_fp32(o, j, I_fx) : orc_vertex_fp64(o, j, I_fx));
            o->fired[j] = (uint8_t)f;
            spikes += (uint64_t)f;
        }
        for (uint32_t j = 0; j < n; ++j)                    /* step 6: record */
            if (o->fired[j]) rast[j >> 5] |= 1u << (j & 31);
        uint64_t delivered = 0;
        int64_t mass_delivered = 0;
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : delivered, mass_delivered)
        for (int64_t jj = 0; jj < (int64_t)n; ++jj) {      /* step 6: deliver */
            if (!o->fired[jj]) continue;
            for (uint64_t e = o->row[jj]; e < o->row[jj + 1]; ++e) {
                int64_t *cell = o->ring + (size_t)((t + o->delay[e]) % D) * n + o->tgt[e];
#pragma omp atomic
                *cell += o->w_fx[e];
                delivered += 1;
                mass_delivered += o->w_fx[e];
            }
        }
        if (o->obs_stride && (t + 1) % o->obs_stride == 0) {   /* step 7: emit one frame */
            const uint64_t frame = (t + 1) / o->obs_stride - 1;
            double *z = o->trace + (size_t)frame * n;
#pragma omp parallel for schedule(static)
            for (int64_t jj = 0; jj < (int64_t)n; ++jj) {
                double sum = o->mode ? (double)o->accf[jj] : o->acc[jj];
                double mean = sum / (double)o->obs_stride;
                double g = o->obs_sigma != 0.0 ? orc_gauss(o->seed, (uint32_t)jj, frame) : 0.0;
                z[jj] = o->obs_gain * mean + o->obs_offset + o->obs_sigma * g;
                o->acc[jj] = 0.0; o->accf[jj] = 0.0f;
            }
            o->frames = frame + 1;
        }
        o->spikes += spikes; o->kicks += kicks; o->delivered += delivered;
        o->mass_consumed += mass_consumed; o->mass_delivered += mass_delivered;
        o->overflow |= overflow;
        o->t = t + 1;
    }
    return o->overflow ? -2 : 0;
}

/* ---- accessors ---------------------------------------------------------------------------- */
enum { ORC_V = 0, ORC_W = 1, ORC_R = 2, ORC_CA = 3, ORC_P = 4, ORC_HM = 5, ORC_HH = 6 };

int orc_get_state(const orc_net *o, int which, double *out)
{
    for (uint32_t j = 0; j < o->n; ++j) {
        switch (which) {
        case ORC_V: out[j] = o->mode ? (double)o->Vf[j] : o->V[j]; break;
        case ORC_W: out[j] = o->mode ? (double)o->Wf[j] : o->W[j]; break;
        case ORC_R: out[j] = o->mode ? (double)o->rf[j] : o->r[j]; break;
        case ORC_CA: out[j] = o->mode ? (double)o->cf[j] : o->c[j]; break;
        case ORC_P: out[j] = o->mode ? (double)o->pf[j] : o->p[j]; break;
        case ORC_HM: out[j] = o->mode ? (double)o->hmf[j] : o->hm[j]; break;
        case ORC_HH: out[j] = o->mode ? (double)o->hhf[j] : o->hh[j]; break;
        default: return -1;
        }
    }
    return 0;
}

int orc_set_state(orc_net *o, int which, const double *in)
{
    for (uint32_t j = 0; j < o->n; ++j) {
        switch (which) {
        case ORC_V: o->V[j] = in[j]; o->Vf[j] = (float)in[j]; break;
        case ORC_W: o->W[j] = in[j]; o->Wf[j] = (float)in[j]; break;
        case ORC_R: o->r[j] = in[j]; o->rf[j] = (float)in[j]; break;
        case ORC_CA: o->c[j] = in[j]; o->cf[j] = (float)in[j]; break;
        case ORC_P: o->p[j] = in[j]; o->pf[j] = (float)in[j]; break;
        case ORC_HM: o->hm[j] = in[j]; o->hmf[j] = (float)in[j]; break;
        case ORC_HH: o->hh[j] = in[j]; o->hhf[j] = (float)in[j]; break;
        default: return -1;
        }
    }
    return 0;
}

void orc_get_refr(const orc_net *o, uint32_t *out) { memcpy(out, o->refr, (size_t)o->n * sizeof(uint32_t)); }
void orc_get_ring(const orc_net *o, int64_t *out) { memcpy(out, o->ring, (size_t)o->D * o->n * sizeof(int64_t)); }
void orc_get_consumed(const orc_net *o, int64_t *out) { memcpy(out, o->consumed, (size_t)o->n * sizeof(int64_t)); }
void orc_get_delays(const orc_net *o, uint32_t *out) { memcpy(out, o->delay, (size_t)o->E * sizeof(uint32_t)); }
void orc_get_w_fx(const orc_net *o, int64_t *out) { memcpy(out, o->w_fx, (size_t)o->E * sizeof(int64_t)); }

int orc_get_raster(const orc_net *o, uint64_t t0, uint64_t n_steps, uint32_t *out)
{
    if (t0 + n_steps > o->t) return -1;
    memcpy(out, o->raster + (size_t)t0 * o->words, (size_t)n_steps * o->words * sizeof(uint32_t));
    return 0;
}

int orc_get_trace(const orc_net *o, uint64_t f0, uint64_t n_frames, double *out)
{
    if (f0 + n_frames > o->frames) return -1;
    memcpy(out, o->trace + (size_t)f0 * o->n, (size_t)n_frames * o->n * sizeof(double));
    return 0;
}

/* out[0..6] = steps, spikes, delivered events, kicks, frames, mass delivered, mass consumed
 * (the two masses are int64 fixed-point sums reinterpreted as uint64). */
void orc_get_counters(const orc_net *o, uint64_t *out)
{
    out[0] = o->t; out[1] = o->spikes; out[2] = o->delivered; out[3] = o->kicks; out[4] = o->frames;
    out[5] = (uint64_t)o->mass_delivered; out[6] = (uint64_t)o->mass_consumed;
}
