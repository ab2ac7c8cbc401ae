/*
 * oracle/fof_oracle_subhalo.c — CPU oracle for the six-dimensional sub-halo pass (SURVEY.md section 8f
 * NEXT-4).  TEST INFRASTRUCTURE, NOT PRODUCT (same rules as fof_oracle.c); shares no code with the
 * CUDA path.
 *
 * PAPER.md:141-154 (section 2.1.1 "Sub-Halo Finding"): "For each identified halo, we then collect the
 * particles associated with it and rerun a second FoF pass that accounts for both particle position
 * x_i and velocity v_i, treating each as a component of a six-dimensional vector", with the metric
 *     d(i,j) = ( (x_i - x_j)^2 / sigma_x + (v_i - v_j)^2 / sigma_v )^(1/2).                  (Eq. 3)
 * Readings (R29-R31; the paper fixes none of them):
 *  R29 two members of one kept halo are linked iff d2 <= ell2, where, all in float32 without FMA,
 *      dx, dy, dz = minimum-image differences of the wrapped positions, dv = plain differences,
 *      d2 = (((dx dx + dy dy) + dz dz) * rx) + (((dvx dvx + dvy dvy) + dvz dvz) * rv),
 *      rx = fl(1 / sigma_x), rv = fl(1 / sigma_v), ell2 = fl(ell * ell)  (ell: the 6-D linking length).
 *  R30 sub_label[i] = minimum original index of i's component in that graph (the same canonical
 *      form as the halo labels); only members of the SAME halo can be linked.
 *  R31 a particle of a dropped halo (particle_group < 0) keeps sub_label[i] = i.
 * The oracle is the definition: all pairs inside each halo, min-label sweeps to the fixed point.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

#define ORACLE_OK 0
#define ORACLE_ERR_ARG (-1)
#define ORACLE_ERR_NOMEM (-3)

int oracle_wrap(const float *pos, int64_t N, float L, float *w); /* fof_oracle.c */

int oracle_link6(const float *wi, const float *vi, const float *wj, const float *vj, float L, float rx, float rv,
                 float ell2)
{
    const float h = 0.5f * L;
    float d[3], u[3];
    for (int k = 0; k < 3; ++k) {
        float dd = wi[k] - wj[k];
        if (dd > h) dd = dd - L;
        else if (dd < -h) dd = dd + L;
        d[k] = dd;
        u[k] = vi[k] - vj[k];
    }
    float xx = d[0] * d[0], yy = d[1] * d[1], zz = d[2] * d[2];
    float sx = xx + yy;
    float dx2 = sx + zz;
    float aa = u[0] * u[0], bb = u[1] * u[1], cc = u[2] * u[2];
    float sv = aa + bb;
    float dv2 = sv + cc;
    float tx = dx2 * rx;
    float tv = dv2 * rv;
    float d2 = tx + tv;
    return d2 <= ell2;
}

static int cmp_pair(const void *a, const void *b)
{
    const int64_t *x = (const int64_t *)a, *y = (const int64_t *)b;
    if (x[0] != y[0]) return x[0] < y[0] ? -1 : 1;
    return (x[1] > y[1]) - (x[1] < y[1]);
}

/* sub_labels [N] written; *E6 = number of linked pairs.  O(sum of squared halo sizes). */
int oracle_subgroups(const float *pos, const float *vel, const int32_t *particle_group, int64_t N, float L,
                     float sigma_x, float sigma_v, float ell, int32_t *sub_labels, uint64_t *E6)
{
    if (N < 0 || !(L > 0.0f) || !(sigma_x > 0.0f) || !(sigma_v > 0.0f) || !(ell > 0.0f)) return ORACLE_ERR_ARG;
    float *w = (float *)malloc(sizeof(float) * 3 * (size_t)(N > 0 ? N : 1));
    int64_t *key = (int64_t *)malloc(sizeof(int64_t) * 2 * (size_t)(N > 0 ? N : 1));
    if (!w || !key) { free(w); free(key); return ORACLE_ERR_NOMEM; }
    int rc = oracle_wrap(pos, N, L, w);
    if (rc) { free(w); free(key); return rc; }
    const float rx = 1.0f / sigma_x, rv = 1.0f / sigma_v, ell2 = ell * ell;
    int64_t m = 0;
    for (int64_t i = 0; i < N; ++i) {
        sub_labels[i] = (int32_t)i;
        if (particle_group[i] >= 0) { key[2 * m] = particle_group[i]; key[2 * m + 1] = i; ++m; }
    }
    qsort(key, (size_t)m, 2 * sizeof(int64_t), cmp_pair);   /* members grouped by halo, ascending index */
    uint64_t E = 0;
    for (int64_t a = 0; a < m;) {
        int64_t b = a;
        while (b < m && key[2 * b] == key[2 * a]) ++b;
        int changed = 1;
        int first = 1;
        while (changed) {            /* min-label sweeps over all pairs of this halo */
            changed = 0;
            for (int64_t p = a; p < b; ++p)
                for (int64_t q = p + 1; q < b; ++q) {
                    const int64_t i = key[2 * p + 1], j = key[2 * q + 1];
                    if (!oracle_link6(w + 3 * i, vel + 3 * i, w + 3 * j, vel + 3 * j, L, rx, rv, ell2)) continue;
                    if (first) ++E;
                    if (sub_labels[i] < sub_labels[j]) { sub_labels[j] = sub_labels[i]; changed = 1; }
                    else if (sub_labels[j] < sub_labels[i]) { sub_labels[i] = sub_labels[j]; changed = 1; }
                }
            first = 0;
        }
        a = b;
    }
    if (E6) *E6 = E;
    free(w); free(key);
    return ORACLE_OK;
}
