/*
 * oracle/fof_oracle_stochastic.c — CPU oracle for stochastic-edge Friends-of-Friends (SURVEY.md
 * section 8f NEXT-3).  TEST INFRASTRUCTURE, NOT PRODUCT (same rules as fof_oracle.c); shares no
 * code with the CUDA path.  Built into the same shared object as fof_oracle.c.
 *
 * What it computes (section 3.2, Eq. 6-8): every potential edge between nearby particles
 * is a Bernoulli variable
 *     y_ij ~ Bernoulli(p_ij),   p_ij = sigma( alpha (b^2 - d_ij^2) / b^2 ),            (Eq. 8)
 * the halos of one Monte Carlo sample are the connected components of the sampled edges, and the
 * REINFORCE estimator (Eq. 7) needs log p(y) = sum_ij [ y log p + (1 - y) log(1 - p) ] and its
 * gradient with respect to the particle positions.
 *
 * Readings (R25-R28; the paper fixes none of these):
 *  R25 potential edges = unordered pairs with float32 minimum-image d2 <= bc2, bc >= b the
 *      candidate radius ("we do not rebuild the neighbor list", section 3.2); pairs beyond
 *      bc have p = 0 and contribute nothing.
 *  R26 sigma ("smooth sigmoidal thresholding function", its form is left open): the logistic
 *      function evaluated by a FIXED float32 recipe so that both sides take the Bernoulli decision
 *      on identical bits:  t = c * (b2 - d2) with c = fl(alpha / b2), clamped to [-30, 30];  z = (-t) * log2(e);
 *      n = rint(z); f = z - n (exact);  2^f by the degree-6 Taylor polynomial in Horner form with
 *      separate multiply and add;  e = 2^f * 2^n (exact scaling);  p = 1 / (1 + e).
 *  R27 randomness: counter-based, 32-bit.  h = mix(fold(seed) ^ (sample * 0x9E3779B9)); h = mix(h + lo);
 *      h = mix(h ^ (hi * 0x85EBCA6B)); u = (h >> 8) * 2^-24, with lo < hi the ORIGINAL indices of the
 *      pair, fold(seed) = low word ^ high word, and mix the 32-bit finaliser
 *      x ^= x >> 16; x *= 0x7FEB352D; x ^= x >> 15; x *= 0x846CA68B; x ^= x >> 16.
 *      y = (u < p).  Independent of traversal order, grid and device.
 *  R28 d log p(y) / d x_i = sum_j (y_ij - p_ij) dt/dx_i,  dt/dx_i = -2 c delta_ij
 *      (delta = minimum-image x_i - x_j), and 0 for a pair whose t was clamped.  float64 sums.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_OK 0
#define ORACLE_ERR_ARG (-1)
#define ORACLE_ERR_NOMEM (-3)

int oracle_wrap(const float *pos, int64_t N, float L, float *w); /* fof_oracle.c */

/* ---- R26: the fixed float32 logistic ----------------------------------------------------------- */
float oracle_sigmoid_fixed(float t)
{
    if (t > 30.0f) t = 30.0f;
    if (t < -30.0f) t = -30.0f;
    const float z = (-t) * 1.44269504088896340736f;
    const float n = rintf(z);                 /* round to nearest even (default rounding mode) */
    const float f = z - n;                    /* |f| <= 0.5, exact */
    float q = 1.5403530393381609954e-4f;      /* ln2^6 / 720 */
    q = q * f; q = q + 1.3333558146428443423e-3f;   /* ln2^5 / 120 */
    q = q * f; q = q + 9.6181291076284771619e-3f;   /* ln2^4 / 24 */
    q = q * f; q = q + 5.5504108664821579953e-2f;   /* ln2^3 / 6 */
    q = q * f; q = q + 2.4022650695910071233e-1f;   /* ln2^2 / 2 */
    q = q * f; q = q + 6.9314718055994530942e-1f;   /* ln2 */
    q = q * f; q = q + 1.0f;
    const float e = ldexpf(q, (int)n);        /* exact: |n| <= 44 */
    return 1.0f / (1.0f + e);
}

/* ---- R27: counter-based uniform, 24 bits ------------------------------------------------------- */
static uint32_t mix32(uint32_t x)
{
    x ^= x >> 16; x *= 0x7FEB352DU;
    x ^= x >> 15; x *= 0x846CA68BU;
    x ^= x >> 16;
    return x;
}

uint32_t oracle_rng_u24(uint64_t seed, uint32_t sample, uint32_t lo, uint32_t hi)
{
    uint32_t h = mix32((uint32_t)(seed ^ (seed >> 32)) ^ (sample * 0x9E3779B9U));   /* per-sample key */
    h = mix32(h + lo);
    h = mix32(h ^ (hi * 0x85EBCA6BU));
    return h >> 8;
}

/* ---- one potential edge: candidate test (R25), p (R26), decision (R27), log-probability term and
 * its gradient with respect to x_i (R28; the gradient with respect to x_j is the negative). ------ */
typedef struct { int cand; int y; float p; double logp; double gi[3]; } pair_term;

static pair_term pair_eval(const float *wi, const float *wj, int32_t i, int32_t j, float L, float bc2, float b2,
                           float alpha, uint64_t seed, uint32_t sample)  /* R26: c = fl(alpha / b2) */
{
    pair_term r;
    memset(&r, 0, sizeof(r));
    const float h = 0.5f * L;
    float d[3];
    for (int k = 0; k < 3; ++k) {
        float dd = wi[k] - wj[k];
        if (dd > h) dd = dd - L;
        else if (dd < -h) dd = dd + L;
        d[k] = dd;
    }
    float xx = d[0] * d[0], yy = d[1] * d[1], zz = d[2] * d[2];
    float s = xx + yy;
    float d2 = s + zz;
    if (!(d2 <= bc2)) return r;
    r.cand = 1;
    float c = alpha / b2;
    float num = b2 - d2;
    float t = c * num;
    r.p = oracle_sigmoid_fixed(t);
    const uint32_t lo = (uint32_t)(i < j ? i : j), hi = (uint32_t)(i < j ? j : i);
    const float u = (float)oracle_rng_u24(seed, sample, lo, hi) * 5.9604644775390625e-8f;  /* 2^-24 */
    r.y = u < r.p;
    r.logp = r.y ? log((double)r.p) : log1p(-(double)r.p);
    if (t <= 30.0f && t >= -30.0f) {
        const double gc = ((double)r.y - (double)r.p) * (-2.0 * (double)c);   /* dt/dx_i = -2 c delta */
        for (int k = 0; k < 3; ++k) r.gi[k] = gc * (double)d[k];
    }
    return r;
}

/* ---- sequential union-find on original indices, root = minimum index ------------- */
static int32_t s_find(int32_t *parent, int32_t x)
{
    int32_t r = x;
    while (parent[r] != r) r = parent[r];
    while (parent[x] != r) { int32_t nx = parent[x]; parent[x] = r; x = nx; }
    return r;
}

static void s_union(int32_t *parent, int32_t a, int32_t c)
{
    int32_t ra = s_find(parent, a), rc = s_find(parent, c);
    if (ra == rc) return;
    if (ra < rc) parent[rc] = ra; else parent[ra] = rc;
}

static void accumulate(const pair_term *t, int32_t i, int32_t j, int32_t *labels, double *logp, double *grad,
                       uint64_t *n_cand, uint64_t *n_edge)
{
    if (!t->cand) return;
    ++*n_cand;
    *logp += t->logp;
    if (grad)
        for (int k = 0; k < 3; ++k) { grad[3 * (int64_t)i + k] += t->gi[k]; grad[3 * (int64_t)j + k] -= t->gi[k]; }
    if (t->y) { ++*n_edge; s_union(labels, i, j); }
}

/* ---- (a) brute force over all i < j: the definition -------------------------------------------
 * labels[i] = minimum original index of i's component in the sampled graph; *logp = log p(y);
 * grad [N,3] (may be NULL) = d log p(y) / d x;  counts of potential and of sampled edges.        */
int oracle_stochastic_brute(const float *pos, int64_t N, float L, float b_cand, float b_link, float alpha,
                            uint64_t seed, uint32_t sample, int32_t *labels, double *logp, double *grad,
                            uint64_t *n_cand, uint64_t *n_edge)
{
    if (N < 0 || !(L > 0.0f) || !(b_link > 0.0f) || !(b_cand >= b_link)) return ORACLE_ERR_ARG;
    float *w = (float *)malloc(sizeof(float) * 3 * (size_t)(N > 0 ? N : 1));
    if (!w) return ORACLE_ERR_NOMEM;
    int rc = oracle_wrap(pos, N, L, w);
    if (rc) { free(w); return rc; }
    const float bc2 = b_cand * b_cand, b2 = b_link * b_link;
    double lp = 0.0;
    uint64_t nc = 0, ne = 0;
    for (int64_t i = 0; i < N; ++i) labels[i] = (int32_t)i;
    if (grad) memset(grad, 0, sizeof(double) * 3 * (size_t)N);
    for (int64_t i = 0; i < N; ++i)
        for (int64_t j = i + 1; j < N; ++j) {
            pair_term t = pair_eval(w + 3 * i, w + 3 * j, (int32_t)i, (int32_t)j, L, bc2, b2, alpha, seed, sample);
            accumulate(&t, (int32_t)i, (int32_t)j, labels, &lp, grad, &nc, &ne);
        }
    for (int64_t i = 0; i < N; ++i) labels[i] = s_find(labels, (int32_t)i);
    if (logp) *logp = lp;
    if (n_cand) *n_cand = nc;
    if (n_edge) *n_edge = ne;
    free(w);
    return ORACLE_OK;
}

/* ---- (b) cell list (own grid: double-precision binning, cell side >= b_cand (1 + 1e-6), at most
 * ~8 N cells, full 27-cell stencil, each unordered pair once): what is used at scale. ------------ */
int oracle_stochastic_cells(const float *pos, int64_t N, float L, float b_cand, float b_link, float alpha,
                            uint64_t seed, uint32_t sample, int32_t *labels, double *logp, double *grad,
                            uint64_t *n_cand, uint64_t *n_edge)
{
    if (N < 0 || N > 2147483647LL || !(L > 0.0f) || !(b_link > 0.0f) || !(b_cand >= b_link)) return ORACLE_ERR_ARG;
    int64_t n = (int64_t)floor((double)L / ((double)b_cand * (1.0 + 1e-6)));
    int64_t lim = 8 * (N > 0 ? N : 1);
    while (n > 3 && n * n * n > lim) --n;
    if (n > 1290) n = 1290;
    if (n < 3)
        return oracle_stochastic_brute(pos, N, L, b_cand, b_link, alpha, seed, sample, labels, logp, grad, n_cand,
                                       n_edge);
    float *w = (float *)malloc(sizeof(float) * 3 * (size_t)(N > 0 ? N : 1));
    int64_t C = n * n * n;
    int32_t *cell = (int32_t *)malloc(sizeof(int32_t) * (size_t)(N > 0 ? N : 1));
    int32_t *start = (int32_t *)calloc((size_t)C + 1, sizeof(int32_t));
    int32_t *order = (int32_t *)malloc(sizeof(int32_t) * (size_t)(N > 0 ? N : 1));
    int32_t *fill = (int32_t *)malloc(sizeof(int32_t) * (size_t)C);
    if (!w || !cell || !start || !order || !fill) {
        free(w); free(cell); free(start); free(order); free(fill);
        return ORACLE_ERR_NOMEM;
    }
    int rc = oracle_wrap(pos, N, L, w);
    if (rc) { free(w); free(cell); free(start); free(order); free(fill); return rc; }
    const float bc2 = b_cand * b_cand, b2 = b_link * b_link;
    double lp = 0.0;
    uint64_t nc = 0, ne = 0;
    for (int64_t i = 0; i < N; ++i) labels[i] = (int32_t)i;
    if (grad) memset(grad, 0, sizeof(double) * 3 * (size_t)N);
    const double s = (double)n / (double)L;
    for (int64_t i = 0; i < N; ++i) {
        int64_t c3[3];
        for (int k = 0; k < 3; ++k) {
            int64_t c = (int64_t)floor((double)w[3 * i + k] * s);
            if (c < 0) c = 0;
            if (c > n - 1) c = n - 1;
            c3[k] = c;
        }
        cell[i] = (int32_t)(c3[0] + n * (c3[1] + n * c3[2]));
        start[cell[i] + 1]++;
    }
    for (int64_t c = 0; c < C; ++c) start[c + 1] += start[c];
    memcpy(fill, start, sizeof(int32_t) * (size_t)C);
    for (int64_t i = 0; i < N; ++i) order[fill[cell[i]]++] = (int32_t)i;
    for (int64_t cz = 0; cz < n; ++cz)
    for (int64_t cy = 0; cy < n; ++cy)
    for (int64_t cx = 0; cx < n; ++cx) {
        const int64_t c = cx + n * (cy + n * cz);
        if (start[c] == start[c + 1]) continue;
        for (int dz = -1; dz <= 1; ++dz)
        for (int dy = -1; dy <= 1; ++dy)
        for (int dx = -1; dx <= 1; ++dx) {
            const int64_t mx = (cx + dx + n) % n, my = (cy + dy + n) % n, mz = (cz + dz + n) % n;
            const int64_t m = mx + n * (my + n * mz);
            for (int32_t p = start[c]; p < start[c + 1]; ++p) {
                const int32_t i = order[p];
                for (int32_t q = start[m]; q < start[m + 1]; ++q) {
                    const int32_t j = order[q];
                    if (i >= j) continue;
                    pair_term t = pair_eval(w + 3 * (int64_t)i, w + 3 * (int64_t)j, i, j, L, bc2, b2, alpha, seed,
                                            sample);
                    accumulate(&t, i, j, labels, &lp, grad, &nc, &ne);
                }
            }
        }
    }
    for (int64_t i = 0; i < N; ++i) labels[i] = s_find(labels, (int32_t)i);
    if (logp) *logp = lp;
    if (n_cand) *n_cand = nc;
    if (n_edge) *n_edge = ne;
    free(w); free(cell); free(start); free(order); free(fill);
    return ORACLE_OK;
}

/* ---- the potential edges of one sample, listed (tiny inputs only; used by the pins) -----------
 * ij [cap,2], y [cap], p [cap]; returns the number of potential edges (may exceed cap).          */
int64_t oracle_stochastic_edges(const float *pos, int64_t N, float L, float b_cand, float b_link, float alpha,
                                uint64_t seed, uint32_t sample, int64_t cap, int32_t *ij, int32_t *y, float *p)
{
    if (N < 0 || !(L > 0.0f) || !(b_link > 0.0f) || !(b_cand >= b_link)) return ORACLE_ERR_ARG;
    float *w = (float *)malloc(sizeof(float) * 3 * (size_t)(N > 0 ? N : 1));
    if (!w) return ORACLE_ERR_NOMEM;
    int rc = oracle_wrap(pos, N, L, w);
    if (rc) { free(w); return rc; }
    const float bc2 = b_cand * b_cand, b2 = b_link * b_link;
    int64_t k = 0;
    for (int64_t i = 0; i < N; ++i)
        for (int64_t j = i + 1; j < N; ++j) {
            pair_term t = pair_eval(w + 3 * i, w + 3 * j, (int32_t)i, (int32_t)j, L, bc2, b2, alpha, seed, sample);
            if (!t.cand) continue;
            if (k < cap) { ij[2 * k] = (int32_t)i; ij[2 * k + 1] = (int32_t)j; y[k] = t.y; p[k] = t.p; }
            ++k;
        }
    free(w);
    return k;
}
