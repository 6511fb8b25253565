/*
 * gn_inputs.c -- seeded synthetic INPUT generator (geometry, graph, weights, classes).
 *
 * This module produces inputs only.  It holds none of the method's arithmetic: no
 * delays (eq. 25), no weight quantisation, no vertex dynamics, no
 * drive/noise generator.  Both the CPU oracle (oracle/) and the CUDA library
 * (paper_0908_3934_b200/) are fed the arrays made here; neither imports the other.
 *
 * Recipe: the paper's workloads are geometric cellular
 * networks (section 3.5, Table 1) which are not available offline;
 * BASELINE.json's distance-probability geometric graphs stand in for them.
 *
 *   positions : uniform in [0, side)^dim, fp32            stream 1, keyed (vertex, axis)
 *   class     : Bernoulli(frac_inh) per vertex            stream 2, keyed (vertex)
 *   edge i->j : i != j, dist < radius, u(i,j) < p(dist)   stream 3, keyed ordered pair (i, j)
 *               kind 0: p = p0            kind 1: p = p0 * exp(-dist / lambda)
 *   weight    : fp32  lo + (hi - lo) * u(i,j), range by the SOURCE's class
 *                                                         stream 4, keyed ordered pair (i, j)
 *   CSR by source, targets ascending inside a row.
 *
 * Randomness is a stateless 64-bit mixing hash of (seed, stream, a, b), so the result does
 * not depend on thread count or visiting order.  Vertex indices inside the keys are LOCAL
 * to a network; batched inputs use one derived seed per network.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC -o libgn_inputs.so gn_inputs.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

static inline uint64_t gni_mix64(uint64_t z)
{
    z += 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

static inline uint64_t gni_hash(uint64_t seed, uint64_t stream, uint64_t a, uint64_t b)
{
    uint64_t h = gni_mix64(seed ^ (stream * 0xD6E8FEB86659FD93ull));
    h = gni_mix64(h ^ a);
    h = gni_mix64(h ^ (b + 0x632BE59BD9B4E019ull));
    return h;
}

/* uniform in [0,1) with 53 bits */
static inline double gni_u01(uint64_t seed, uint64_t stream, uint64_t a, uint64_t b)
{
    return (double)(gni_hash(seed, stream, a, b) >> 11) * (1.0 / 9007199254740992.0);
}

uint64_t gni_derive_seed(uint64_t seed, uint64_t index)
{
    return gni_hash(seed, 7, index, 0);
}

void gni_positions(uint64_t seed, uint32_t n, uint32_t dim, double side, float *pos)
{
    for (uint32_t i = 0; i < n; ++i)
        for (uint32_t k = 0; k < dim; ++k) {
            float x = (float)(side * gni_u01(seed, 1, i, k));
            if (x >= (float)side) x = nextafterf((float)side, 0.0f);
            pos[(size_t)i * dim + k] = x;
        }
}

void gni_classes(uint64_t seed, uint32_t n, double frac_inh, uint8_t *cls)
{
    for (uint32_t i = 0; i < n; ++i)
        cls[i] = gni_u01(seed, 2, i, 0) < frac_inh ? 1 : 0;
}

/* ---- cell list over one network --------------------------------------------------- */
typedef struct {
    uint32_t nc;          /* cells per axis */
    double inv_cell;
    uint32_t *cell_start; /* [ncells + 1] */
    uint32_t *cell_items; /* [n] vertex ids sorted by cell (ascending id inside a cell) */
} gni_cells;

static uint32_t gni_cell_of(const gni_cells *c, const float *p, uint32_t dim)
{
    uint32_t idx = 0;
    for (uint32_t k = dim; k-- > 0;) {
        int32_t q = (int32_t)((double)p[k] * c->inv_cell);
        if (q < 0) q = 0;
        if ((uint32_t)q >= c->nc) q = (int32_t)c->nc - 1;
        idx = idx * c->nc + (uint32_t)q;
    }
    return idx;
}

static int gni_cells_build(gni_cells *c, const float *pos, uint32_t n, uint32_t dim, double side,
                           double radius)
{
    /* cell edge = radius / sub, sub in {3,2,1}: the finest grid that still holds >= 2 vertices per cell */
    uint32_t nc = 1;
    for (uint32_t sub = 3; sub >= 1; --sub) {
        nc = (uint32_t)floor(side * (double)sub / radius);
        if (nc < 1) nc = 1;
        if (nc > 1024) nc = 1024;
        double ncells_d = pow((double)nc, (double)dim);
        if ((double)n / ncells_d >= 2.0 || sub == 1) break;
    }
    c->nc = nc;
    c->inv_cell = (double)nc / side;
    size_t ncells = 1;
    for (uint32_t k = 0; k < dim; ++k) ncells *= nc;
    c->cell_start = (uint32_t *)calloc(ncells + 1, sizeof(uint32_t));
    c->cell_items = (uint32_t *)malloc((size_t)(n ? n : 1) * sizeof(uint32_t));
    if (!c->cell_start || !c->cell_items) return -1;
    for (uint32_t i = 0; i < n; ++i) c->cell_start[gni_cell_of(c, pos + (size_t)i * dim, dim) + 1]++;
    for (size_t k = 0; k < ncells; ++k) c->cell_start[k + 1] += c->cell_start[k];
    uint32_t *fill = (uint32_t *)malloc(ncells * sizeof(uint32_t));
    if (!fill) return -1;
    memcpy(fill, c->cell_start, ncells * sizeof(uint32_t));
    for (uint32_t i = 0; i < n; ++i) c->cell_items[fill[gni_cell_of(c, pos + (size_t)i * dim, dim)]++] = i;
    free(fill);
    return 0;
}

static void gni_cells_free(gni_cells *c)
{
    free(c->cell_start);
    free(c->cell_items);
}

typedef struct {
    uint32_t kind; /* 0: constant p0 inside radius; 1: p0 * exp(-d/lambda) inside radius */
    double radius, p0, lambda;
} gni_rule;

static int gni_cmp_u32(const void *a, const void *b)
{
    uint32_t x = *(const uint32_t *)a, y = *(const uint32_t *)b;
    return (x > y) - (x < y);
}

/* Collect the out-neighbours of local vertex i into out[] (ascending); returns the count.
 * out may be NULL (count only). */
static uint32_t gni_row(const gni_cells *c, const float *pos, uint32_t dim, const gni_rule *rule,
                        uint64_t seed, uint32_t i, uint32_t *out)
{
    const float *pi = pos + (size_t)i * dim;
    const double r2 = rule->radius * rule->radius;
    uint32_t cnt = 0;
    int32_t lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0};
    for (uint32_t k = 0; k < dim; ++k) {
        /* every cell the ball of `radius` around vertex i can touch (one cell of slack for rounding) */
        lo[k] = (int32_t)floor(((double)pi[k] - rule->radius) * c->inv_cell) - 1;
        hi[k] = (int32_t)floor(((double)pi[k] + rule->radius) * c->inv_cell) + 1;
        if (lo[k] < 0) lo[k] = 0;
        if (hi[k] > (int32_t)c->nc - 1) hi[k] = (int32_t)c->nc - 1;
    }
    for (int32_t z = lo[2]; z <= hi[2]; ++z)
        for (int32_t y = lo[1]; y <= hi[1]; ++y)
            for (int32_t x = lo[0]; x <= hi[0]; ++x) {
                size_t cell = ((size_t)z * c->nc + (size_t)y) * c->nc + (size_t)x;
                if (dim == 2) cell = (size_t)y * c->nc + (size_t)x;
                for (uint32_t s = c->cell_start[cell]; s < c->cell_start[cell + 1]; ++s) {
                    uint32_t j = c->cell_items[s];
                    if (j == i) continue;
                    const float *pj = pos + (size_t)j * dim;
                    double d2 = 0.0;
                    for (uint32_t k = 0; k < dim; ++k) {
                        double d = (double)pi[k] - (double)pj[k];
                        d2 += d * d;
                    }
                    if (!(d2 < r2)) continue;
                    double u = gni_u01(seed, 3, i, j);
                    if (!(u < rule->p0)) continue;
                    if (rule->kind == 1 && !(u < rule->p0 * exp(-sqrt(d2) / rule->lambda))) continue;
                    if (out) out[cnt] = j;
                    ++cnt;
                }
            }
    if (out && cnt > 1) qsort(out, cnt, sizeof(uint32_t), gni_cmp_u32);
    return cnt;
}

/*
 * Pass 1: out-degree of every vertex of `n_networks` networks of `n_per` vertices each
 * (positions concatenated, seeds[b] per network).  degree[] has n_networks * n_per entries.
 */
int gni_degrees(uint32_t n_networks, uint32_t n_per, uint32_t dim, double side, const float *pos,
                uint32_t kind, double radius, double p0, double lambda, const uint64_t *seeds,
                uint32_t *degree)
{
    gni_rule rule = {kind, radius, p0, lambda};
    int err = 0;
    if (n_networks == 1) {
        gni_cells c;
        if (gni_cells_build(&c, pos, n_per, dim, side, radius)) return -1;
#pragma omp parallel for schedule(dynamic, 256)
        for (int64_t i = 0; i < (int64_t)n_per; ++i)
            degree[i] = gni_row(&c, pos, dim, &rule, seeds[0], (uint32_t)i, NULL);
        gni_cells_free(&c);
        return 0;
    }
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t b = 0; b < (int64_t)n_networks; ++b) {
        const float *p = pos + (size_t)b * n_per * dim;
        gni_cells c;
        if (gni_cells_build(&c, p, n_per, dim, side, radius)) {
            err = -1;
            continue;
        }
        for (uint32_t i = 0; i < n_per; ++i)
            degree[(size_t)b * n_per + i] = gni_row(&c, p, dim, &rule, seeds[b], i, NULL);
        gni_cells_free(&c);
    }
    return err;
}

/*
 * Pass 2: fill targets (GLOBAL vertex ids = network offset + local id) and fp32 weights.
 * row_offsets[] is the exclusive prefix sum of degree[] (n_networks * n_per + 1 entries).
 * w_range = { exc_lo, exc_hi, inh_lo, inh_hi }: weight range by the source's class.
 */
int gni_fill(uint32_t n_networks, uint32_t n_per, uint32_t dim, double side, const float *pos,
             uint32_t kind, double radius, double p0, double lambda, const uint64_t *seeds,
             const uint8_t *cls, const double *w_range, const uint64_t *row_offsets,
             uint32_t *targets, float *weights)
{
    gni_rule rule = {kind, radius, p0, lambda};
    int err = 0;
    if (n_networks == 1) {
        gni_cells c;
        if (gni_cells_build(&c, pos, n_per, dim, side, radius)) return -1;
#pragma omp parallel for schedule(dynamic, 256)
        for (int64_t i = 0; i < (int64_t)n_per; ++i) {
            uint32_t *row = targets + row_offsets[i];
            uint32_t cnt = gni_row(&c, pos, dim, &rule, seeds[0], (uint32_t)i, row);
            if ((uint64_t)cnt != row_offsets[i + 1] - row_offsets[i]) err = -2;
            const double lo = w_range[cls[i] ? 2 : 0], hi = w_range[cls[i] ? 3 : 1];
            for (uint32_t e = 0; e < cnt; ++e)
                weights[row_offsets[i] + e] = (float)(lo + (hi - lo) * gni_u01(seeds[0], 4, (uint64_t)i, row[e]));
        }
        gni_cells_free(&c);
        return err;
    }
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t b = 0; b < (int64_t)n_networks; ++b) {
        const float *p = pos + (size_t)b * n_per * dim;
        const uint32_t base = (uint32_t)((size_t)b * n_per);
        gni_cells c;
        if (gni_cells_build(&c, p, n_per, dim, side, radius)) {
            err = -1;
            continue;
        }
        for (uint32_t i = 0; i < n_per; ++i) {
            const uint64_t r0 = row_offsets[(size_t)base + i];
            uint32_t *row = targets + r0;
            uint32_t cnt = gni_row(&c, p, dim, &rule, seeds[b], i, row);
            if ((uint64_t)cnt != row_offsets[(size_t)base + i + 1] - r0) err = -2;
            const uint8_t ci = cls[(size_t)base + i];
            const double lo = w_range[ci ? 2 : 0], hi = w_range[ci ? 3 : 1];
            for (uint32_t e = 0; e < cnt; ++e) {
                weights[r0 + e] = (float)(lo + (hi - lo) * gni_u01(seeds[b], 4, (uint64_t)i, row[e]));
                row[e] += base;
            }
        }
        gni_cells_free(&c);
    }
    return err;
}
