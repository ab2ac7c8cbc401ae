/*
 * oracle/fof_oracle.c — CPU oracle for periodic Friends-of-Friends linking.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.  It shares no code,
 * header, table or helper with the CUDA path under paper_2510_26851_b200/csrc/.
 *
 * Plain, slow, obviously-correct C99, written from the paper (PAPER.md = /root/reference/PAPER.md
 * at survey time; not read at run time):
 *   - what is linked: PAPER.md:85-87 (§2 step iv), PAPER.md:210-214 (Alg. 2 mask: minimum-image
 *     ||Delta_ij|| <= b), PAPER.md:160 ("exact equivalence with the canonical FoF connectivity
 *     criterion");
 *   - labels: fixed point of min-label propagation with l_i initialised to i, PAPER.md:66 (step i),
 *     PAPER.md:89-91 (step v), PAPER.md:221-225 (Alg. 2 "Label propagation");
 *   - compaction and sizes: PAPER.md:93-95 (step vi), PAPER.md:227 (Alg. 2 "Compaction");
 *   - halo position: PAPER.md:259 (Eq. 4, plain mean), made periodic per DESIGN.md reading R11.
 * Readings of silent / ambiguous points are the ones listed in DESIGN.md §3 (R1..R17).
 *
 * Build:  gcc -O2 -std=c99 -ffp-contract=off -fno-fast-math -shared -fPIC fof_oracle.c -lm
 *         (-ffp-contract=off: the link predicate is float32 with NO fused multiply-add.)
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): dyadic hand cases for the predicate; brute force
 * (a) vs cell list (b); scipy connected_components; float64 cKDTree sandwich; lattice / planted
 * cliques / chain / Poisson closed forms; permutation and translation invariance; numpy
 * unique/bincount for groups; Eq. 4 plain mean for the centre of mass.
 * Parity unpinned: agreement with the paper's own fastPM + cFoF catalogs —
 * neither data nor code is available and the paper prints no values.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_OK 0
#define ORACLE_ERR_ARG (-1)
#define ORACLE_ERR_NONFINITE (-2)
#define ORACLE_ERR_NOMEM (-3)

/* ---- step 1: wrap into [0, L)  ("X <- X mod L"; R6) ------------------ */
float oracle_wrap1(float x, float L)
{
    if (x >= 0.0f && x < L) return x;
    float t = x / L;
    float f = floorf(t);
    float p = L * f;          /* rounded product: no FMA (-ffp-contract=off) */
    float w = x - p;
    if (w < 0.0f) w = w + L;
    if (!(w >= 0.0f) || w >= L) w = 0.0f;  /* R6: |x| beyond ~2^24 L, where x - L floor(x/L) is off by whole ulps of x */
    return w;
}

int oracle_wrap(const float *pos, int64_t N, float L, float *w)
{
    if (N < 0 || !(L > 0.0f)) return ORACLE_ERR_ARG;
    for (int64_t i = 0; i < 3 * N; ++i) {
        if (!isfinite(pos[i])) return ORACLE_ERR_NONFINITE;
        w[i] = oracle_wrap1(pos[i], L);
    }
    return ORACLE_OK;
}

/* ---- step 2: link predicate (expression fixed by north_star, R1/R7) -----
 * all float32, round to nearest, no FMA:  per axis d = wi - wj; if d > h: d -= L; else if d < -h:
 * d += L;  d2 = (dx*dx + dy*dy) + dz*dz;  link <=> d2 <= b2,  h = 0.5 L, b2 = fl(b*b).          */
int oracle_link(const float *wi, const float *wj, float L, float b)
{
    const float h = 0.5f * L;
    const float b2 = b * b;
    float d[3];
    for (int k = 0; k < 3; ++k) {
        float dd = wi[k] - wj[k];
        if (dd > h) dd = dd - L;
        else if (dd < -h) dd = dd + L;
        d[k] = dd;
    }
    float xx = d[0] * d[0];
    float yy = d[1] * d[1];
    float zz = d[2] * d[2];
    float s = xx + yy;
    float d2 = s + zz;
    return d2 <= b2;
}

/* ---- (a) brute force: all pairs + the paper's min-label sweeps until nothing changes ----------
 * "Initialize l_i <- i. for t <- 1..T: for all edges (i<->j): l_i <- min(l_i,l_j)
 * and l_j <- min(l_j, l_i)".  T is replaced by "until a sweep changes nothing" (R4), whose fixed
 * point is label = minimum index of the connected component.                      */
int oracle_labels_brute(const float *pos, int64_t N, float L, float b, int32_t *labels, uint64_t *E_out)
{
    if (N < 0 || !(L > 0.0f) || !(b > 0.0f)) return ORACLE_ERR_ARG;
    float *w = (float *)malloc(sizeof(float) * 3 * (size_t)(N > 0 ? N : 1));
    if (!w) return ORACLE_ERR_NOMEM;
    int rc = oracle_wrap(pos, N, L, w);
    if (rc) { free(w); return rc; }
    /* edge list */
    size_t cap = 1024, ne = 0;
    int32_t *ei = (int32_t *)malloc(cap * sizeof(int32_t));
    int32_t *ej = (int32_t *)malloc(cap * sizeof(int32_t));
    if (!ei || !ej) { free(w); free(ei); free(ej); return ORACLE_ERR_NOMEM; }
    for (int64_t i = 0; i < N; ++i)
        for (int64_t j = i + 1; j < N; ++j)
            if (oracle_link(w + 3 * i, w + 3 * j, L, b)) {
                if (ne == cap) {
                    cap *= 2;
                    ei = (int32_t *)realloc(ei, cap * sizeof(int32_t));
                    ej = (int32_t *)realloc(ej, cap * sizeof(int32_t));
                    if (!ei || !ej) { free(w); free(ei); free(ej); return ORACLE_ERR_NOMEM; }
                }
                ei[ne] = (int32_t)i; ej[ne] = (int32_t)j; ++ne;
            }
    for (int64_t i = 0; i < N; ++i) labels[i] = (int32_t)i;
    int changed = 1;
    while (changed) {
        changed = 0;
        for (size_t e = 0; e < ne; ++e) {
            int32_t a = labels[ei[e]], c = labels[ej[e]];
            if (a < c) { labels[ej[e]] = a; changed = 1; }
            else if (c < a) { labels[ei[e]] = c; changed = 1; }
        }
    }
    if (E_out) *E_out = (uint64_t)ne;
    free(w); free(ei); free(ej);
    return ORACLE_OK;
}

/* ---- (b) cell list + sequential union-find (what is used and timed at scale) ------------------
 * Own grid: double-precision binning, n = floor(L / (b (1 + 1e-6))) per axis, coarsened until
 * n^3 <= 8 N; full 27-cell stencil with indices mod n; each unordered particle
 * pair tested once (i < j).  n < 3 -> every pair is tested (the stencil would alias).           */
static int32_t uf_find(int32_t *parent, int32_t x)
{
    int32_t r = x;
    while (parent[r] != r) r = parent[r];
    while (parent[x] != r) { int32_t nx = parent[x]; parent[x] = r; x = nx; }
    return r;
}

static void uf_union(int32_t *parent, int32_t a, int32_t c)
{
    int32_t ra = uf_find(parent, a), rc = uf_find(parent, c);
    if (ra == rc) return;
    if (ra < rc) parent[rc] = ra; else parent[ra] = rc;   /* root = minimum index */
}

static int64_t oracle_grid_n(int64_t N, float L, float b)
{
    int64_t n = (int64_t)floor((double)L / ((double)b * (1.0 + 1e-6)));
    if (n < 1) n = 1;
    int64_t lim = 8 * (N > 0 ? N : 1);
    while (n > 3 && n * n * n > lim) --n;
    if (n > 1290) n = 1290;   /* n^3 < 2^31 */
    return n;
}

int oracle_labels_cells(const float *pos, int64_t N, float L, float b, int32_t *labels, uint64_t *E_out)
{
    if (N < 0 || N > 2147483647LL || !(L > 0.0f) || !(b > 0.0f)) return ORACLE_ERR_ARG;
    float *w = (float *)malloc(sizeof(float) * 3 * (size_t)(N > 0 ? N : 1));
    if (!w) return ORACLE_ERR_NOMEM;
    int rc = oracle_wrap(pos, N, L, w);
    if (rc) { free(w); return rc; }
    for (int64_t i = 0; i < N; ++i) labels[i] = (int32_t)i;
    uint64_t E = 0;
    int64_t n = oracle_grid_n(N, L, b);
    if (n < 3) {
        for (int64_t i = 0; i < N; ++i)
            for (int64_t j = i + 1; j < N; ++j)
                if (oracle_link(w + 3 * i, w + 3 * j, L, b)) { ++E; uf_union(labels, (int32_t)i, (int32_t)j); }
    } else {
        int64_t C = n * n * n;
        int32_t *cell = (int32_t *)malloc(sizeof(int32_t) * (size_t)(N > 0 ? N : 1));
        int32_t *start = (int32_t *)calloc((size_t)C + 1, sizeof(int32_t));
        int32_t *order = (int32_t *)malloc(sizeof(int32_t) * (size_t)(N > 0 ? N : 1));
        if (!cell || !start || !order) { free(w); free(cell); free(start); free(order); return ORACLE_ERR_NOMEM; }
        double s = (double)n / (double)L;
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
        int32_t *fill = (int32_t *)malloc(sizeof(int32_t) * (size_t)C);
        if (!fill) { free(w); free(cell); free(start); free(order); return ORACLE_ERR_NOMEM; }
        memcpy(fill, start, sizeof(int32_t) * (size_t)C);
        for (int64_t i = 0; i < N; ++i) order[fill[cell[i]]++] = (int32_t)i;
        free(fill);
        for (int64_t cz = 0; cz < n; ++cz)
        for (int64_t cy = 0; cy < n; ++cy)
        for (int64_t cx = 0; cx < n; ++cx) {
            int64_t c = cx + n * (cy + n * cz);
            if (start[c] == start[c + 1]) continue;
            for (int dz = -1; dz <= 1; ++dz)
            for (int dy = -1; dy <= 1; ++dy)
            for (int dx = -1; dx <= 1; ++dx) {
                int64_t mx = (cx + dx + n) % n, my = (cy + dy + n) % n, mz = (cz + dz + n) % n;
                int64_t m = mx + n * (my + n * mz);
                for (int32_t p = start[c]; p < start[c + 1]; ++p) {
                    int32_t i = order[p];
                    for (int32_t q = start[m]; q < start[m + 1]; ++q) {
                        int32_t j = order[q];
                        if (i < j && oracle_link(w + 3 * (int64_t)i, w + 3 * (int64_t)j, L, b)) {
                            ++E;
                            uf_union(labels, i, j);
                        }
                    }
                }
            }
        }
        free(cell); free(start); free(order);
    }
    for (int64_t i = 0; i < N; ++i) labels[i] = uf_find(labels, (int32_t)i);
    if (E_out) *E_out = E;
    free(w);
    return ORACLE_OK;
}

/* ---- the same linker with the PAIR SEARCH on several host threads ("a second figure with the
 * pair search OpenMP-parallel over cell slabs (per-thread edge buffers, serial union) on all host cores, labels
 * required identical to the single-thread oracle").  Same grid, same stencil, same predicate, same union-find;
 * only the order in which the edges reach the union-find differs, and the root of a set is its minimum index
 * whatever that order is.  It exists for the all-cores CPU figure of bench.py; parity uses oracle_labels_cells. */
typedef struct { int32_t i, j; } edge_t;

int oracle_labels_cells_threads(const float *pos, int64_t N, float L, float b, int32_t *labels, uint64_t *E_out,
                                int32_t threads)
{
    if (N < 0 || N > 2147483647LL || !(L > 0.0f) || !(b > 0.0f) || threads < 1) return ORACLE_ERR_ARG;
    int64_t n = oracle_grid_n(N, L, b);
    if (n < 3) return oracle_labels_cells(pos, N, L, b, labels, E_out);
    float *w = (float *)malloc(sizeof(float) * 3 * (size_t)(N > 0 ? N : 1));
    if (!w) return ORACLE_ERR_NOMEM;
    int rc = oracle_wrap(pos, N, L, w);
    if (rc) { free(w); return rc; }
    for (int64_t i = 0; i < N; ++i) labels[i] = (int32_t)i;
    int64_t C = n * n * n;
    int32_t *cell = (int32_t *)malloc(sizeof(int32_t) * (size_t)(N > 0 ? N : 1));
    int32_t *start = (int32_t *)calloc((size_t)C + 1, sizeof(int32_t));
    int32_t *order = (int32_t *)malloc(sizeof(int32_t) * (size_t)(N > 0 ? N : 1));
    int32_t *fill = (int32_t *)malloc(sizeof(int32_t) * (size_t)C);
    edge_t **ebuf = (edge_t **)calloc((size_t)n, sizeof(edge_t *));   /* one edge buffer per z slab of cells */
    int64_t *ecnt = (int64_t *)calloc((size_t)n, sizeof(int64_t));
    if (!cell || !start || !order || !fill || !ebuf || !ecnt) {
        free(w); free(cell); free(start); free(order); free(fill); free(ebuf); free(ecnt);
        return ORACLE_ERR_NOMEM;
    }
    double s = (double)n / (double)L;
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
    free(fill);
    int failed = 0;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(threads)
#endif
    for (int64_t cz = 0; cz < n; ++cz) {
        int64_t capz = 1024, cnt = 0;
        edge_t *buf = (edge_t *)malloc(sizeof(edge_t) * (size_t)capz);
        for (int64_t cy = 0; cy < n && buf; ++cy)
        for (int64_t cx = 0; cx < n && buf; ++cx) {
            int64_t c = cx + n * (cy + n * cz);
            if (start[c] == start[c + 1]) continue;
            for (int dz = -1; dz <= 1; ++dz)
            for (int dy = -1; dy <= 1; ++dy)
            for (int dx = -1; dx <= 1; ++dx) {
                int64_t mx = (cx + dx + n) % n, my = (cy + dy + n) % n, mz = (cz + dz + n) % n;
                int64_t m = mx + n * (my + n * mz);
                for (int32_t p = start[c]; p < start[c + 1] && buf; ++p) {
                    int32_t i = order[p];
                    for (int32_t q = start[m]; q < start[m + 1]; ++q) {
                        int32_t j = order[q];
                        if (i < j && oracle_link(w + 3 * (int64_t)i, w + 3 * (int64_t)j, L, b)) {
                            if (cnt == capz) {
                                capz *= 2;
                                edge_t *nb = (edge_t *)realloc(buf, sizeof(edge_t) * (size_t)capz);
                                if (!nb) { free(buf); buf = NULL; break; }
                                buf = nb;
                            }
                            buf[cnt].i = i; buf[cnt].j = j; ++cnt;
                        }
                    }
                }
            }
        }
        if (!buf) {
#ifdef _OPENMP
#pragma omp atomic write
#endif
            failed = 1;
        }
        ebuf[cz] = buf;
        ecnt[cz] = buf ? cnt : 0;
    }
    uint64_t E = 0;
    for (int64_t cz = 0; cz < n; ++cz) {          /* the serial union step */
        for (int64_t k = 0; k < ecnt[cz]; ++k) uf_union(labels, ebuf[cz][k].i, ebuf[cz][k].j);
        E += (uint64_t)ecnt[cz];
        free(ebuf[cz]);
    }
    for (int64_t i = 0; i < N; ++i) labels[i] = uf_find(labels, (int32_t)i);
    if (E_out) *E_out = E;
    free(w); free(cell); free(start); free(order); free(ebuf); free(ecnt);
    return failed ? ORACLE_ERR_NOMEM : ORACLE_OK;
}

/* ---- groups (Eq. 4 PAPER.md:259 made periodic, R9-R13) ----------
 * distinct labels ascending; size = member count; keep size >= N_min; kept groups numbered 0..K-1
 * by ascending canonical label.  mass = sum m_i in float64.  centre of mass: r = w[label];
 * delta_i = (double)w_i - (double)r per axis with the +-L/2 select in double;
 * com = r + sum m_i delta_i / sum m_i, wrapped into [0, L).
 * Outputs have capacity `cap`; returns K (>= 0) or a negative error; K > cap -> ORACLE_ERR_ARG.  */
int64_t oracle_groups(const float *pos, const float *mass, const int32_t *labels, int64_t N, float L,
                      int32_t N_min, int64_t cap, int32_t *group_label, int32_t *group_size,
                      double *group_mass, double *group_com, int32_t *particle_group)
{
    if (N < 0 || !(L > 0.0f) || N_min < 1) return ORACLE_ERR_ARG;
    float *w = (float *)malloc(sizeof(float) * 3 * (size_t)(N > 0 ? N : 1));
    int32_t *size = (int32_t *)calloc((size_t)(N > 0 ? N : 1), sizeof(int32_t));
    int32_t *gid = (int32_t *)malloc(sizeof(int32_t) * (size_t)(N > 0 ? N : 1));
    if (!w || !size || !gid) { free(w); free(size); free(gid); return ORACLE_ERR_NOMEM; }
    int rc = oracle_wrap(pos, N, L, w);
    if (rc) { free(w); free(size); free(gid); return rc; }
    for (int64_t i = 0; i < N; ++i) {
        if (labels[i] < 0 || labels[i] >= N) { free(w); free(size); free(gid); return ORACLE_ERR_ARG; }
        size[labels[i]]++;
    }
    int64_t K = 0;
    for (int64_t g = 0; g < N; ++g) {
        gid[g] = -1;
        if (size[g] >= N_min) {
            if (K < cap) { group_label[K] = (int32_t)g; group_size[K] = size[g]; }
            gid[g] = (int32_t)K;
            ++K;
        }
    }
    if (K > cap) { free(w); free(size); free(gid); return ORACLE_ERR_ARG; }
    double *sm = (double *)calloc((size_t)(K > 0 ? K : 1) * 4, sizeof(double));
    if (!sm) { free(w); free(size); free(gid); return ORACLE_ERR_NOMEM; }
    const double Ld = (double)L, hd = 0.5 * (double)L;
    for (int64_t i = 0; i < N; ++i) {
        int32_t k = gid[labels[i]];
        if (particle_group) particle_group[i] = k;
        if (k < 0) continue;
        double m = mass ? (double)mass[i] : 1.0;
        const float *r = w + 3 * (int64_t)labels[i];
        sm[4 * k + 3] += m;
        for (int a = 0; a < 3; ++a) {
            double d = (double)w[3 * i + a] - (double)r[a];
            if (d > hd) d = d - Ld; else if (d < -hd) d = d + Ld;
            sm[4 * k + a] += m * d;
        }
    }
    for (int64_t k = 0; k < K; ++k) {
        const float *r = w + 3 * (int64_t)group_label[k];
        group_mass[k] = sm[4 * k + 3];
        for (int a = 0; a < 3; ++a) {
            double c = (double)r[a] + sm[4 * k + a] / sm[4 * k + 3];
            if (c < 0.0) c += Ld;
            if (c >= Ld) c -= Ld;
            group_com[3 * k + a] = c;
        }
    }
    free(w); free(size); free(gid); free(sm);
    return K;
}

/* ---- NEXT-1: halo decoration and frozen-assignment backward ------------------
 * PAPER.md:255-261 (section 3.1 "Frozen Assignment", Eq. 4): membership is held fixed and
 *     X^h = (1/N) sum_i x_i   ->   dX^h/dtheta = (1/N) sum_i dx_i/dtheta,
 * i.e. dL/dx_i = (m_i / M_g) dL/dX_g for a member i of group g (mass-weighted as the forward is,
 * DESIGN.md R12) and 0 for a particle of a dropped group.
 * PAPER.md:283-290 (section 3.1.1 "Decorated Frozen Assignment", Eq. 5): the decoration is the
 * "particle standard deviation (sigma)" of a halo.  The paper gives no formula; reading R23
 * (DESIGN.md): sigma_g = sqrt( sum_i m_i |delta_i|^2 / M_g ) with delta_i the minimum-image
 * displacement of member i from the periodic centre of mass X_g, all in float64.  Its derivative
 * at fixed membership is d sigma_g / d x_i = (m_i / (M_g sigma_g)) delta_i (the terms through X_g
 * cancel because sum_i m_i delta_i = 0); it is taken as 0 where sigma_g = 0.
 * Both functions follow the definition with one plain pass over the particles.
 * Pins (tests/test_oracle_next1.py): numpy mean / std for groups away from the box faces,
 * translation across a face, closed forms (unit masses: gradient = G/N_g), and central finite
 * differences of an independent numpy forward.                                                  */
int oracle_group_sigma(const float *pos, const float *mass, const int32_t *particle_group, int64_t N, float L,
                       int64_t K, const double *group_com, double *group_sigma)
{
    if (N < 0 || K < 0 || !(L > 0.0f)) return ORACLE_ERR_ARG;
    float *w = (float *)malloc(sizeof(float) * 3 * (size_t)(N > 0 ? N : 1));
    double *sq = (double *)calloc((size_t)(K > 0 ? K : 1) * 2, sizeof(double));
    if (!w || !sq) { free(w); free(sq); return ORACLE_ERR_NOMEM; }
    int rc = oracle_wrap(pos, N, L, w);
    if (rc) { free(w); free(sq); return rc; }
    const double Ld = (double)L, hd = 0.5 * (double)L;
    for (int64_t i = 0; i < N; ++i) {
        const int32_t k = particle_group[i];
        if (k < 0) continue;
        if (k >= K) { free(w); free(sq); return ORACLE_ERR_ARG; }
        const double m = mass ? (double)mass[i] : 1.0;
        double d2 = 0.0;
        for (int a = 0; a < 3; ++a) {
            double d = (double)w[3 * i + a] - group_com[3 * k + a];
            if (d > hd) d = d - Ld; else if (d < -hd) d = d + Ld;
            d2 += d * d;
        }
        sq[2 * k] += m * d2;
        sq[2 * k + 1] += m;
    }
    for (int64_t k = 0; k < K; ++k) group_sigma[k] = sq[2 * k + 1] > 0.0 ? sqrt(sq[2 * k] / sq[2 * k + 1]) : 0.0;
    free(w); free(sq);
    return ORACLE_OK;
}

int oracle_groups_backward(const float *pos, const float *mass, const int32_t *particle_group, int64_t N, float L,
                           int64_t K, const double *group_mass, const double *group_com,
                           const double *group_sigma, const double *grad_com, const double *grad_sigma,
                           double *grad_pos)
{
    if (N < 0 || K < 0 || !(L > 0.0f)) return ORACLE_ERR_ARG;
    if (grad_sigma && !group_sigma) return ORACLE_ERR_ARG;
    float *w = (float *)malloc(sizeof(float) * 3 * (size_t)(N > 0 ? N : 1));
    if (!w) return ORACLE_ERR_NOMEM;
    int rc = oracle_wrap(pos, N, L, w);
    if (rc) { free(w); return rc; }
    const double Ld = (double)L, hd = 0.5 * (double)L;
    for (int64_t i = 0; i < N; ++i) {
        const int32_t k = particle_group[i];
        for (int a = 0; a < 3; ++a) grad_pos[3 * i + a] = 0.0;
        if (k < 0) continue;
        if (k >= K) { free(w); return ORACLE_ERR_ARG; }
        const double m = mass ? (double)mass[i] : 1.0;
        const double wgt = m / group_mass[k];
        for (int a = 0; a < 3; ++a) {
            double g = grad_com ? wgt * grad_com[3 * k + a] : 0.0;
            if (grad_sigma && group_sigma[k] > 0.0) {
                double d = (double)w[3 * i + a] - group_com[3 * k + a];
                if (d > hd) d = d - Ld; else if (d < -hd) d = d + Ld;
                g += grad_sigma[k] * wgt * d / group_sigma[k];
            }
            grad_pos[3 * i + a] = g;
        }
    }
    free(w);
    return ORACLE_OK;
}

/* ---- P_ref: candidate pairs of the linked-cell method on the tightest grid n_ref = floor(L/b) ---
 * (27-cell stencil, each unordered particle pair counted once).  Metric denominator only
 * (DESIGN.md §6); sorted keys + run lengths, no dense cell array.                               */
static int cmp_i64(const void *a, const void *c)
{
    int64_t x = *(const int64_t *)a, y = *(const int64_t *)c;
    return (x > y) - (x < y);
}

static int64_t occ_of(const int64_t *keys, const int64_t *cnt, int64_t U, int64_t key)
{
    int64_t lo = 0, hi = U;
    while (lo < hi) { int64_t mid = (lo + hi) / 2; if (keys[mid] < key) lo = mid + 1; else hi = mid; }
    return (lo < U && keys[lo] == key) ? cnt[lo] : 0;
}

int oracle_pref(const float *pos, int64_t N, float L, float b, uint64_t *P_out)
{
    if (N < 0 || !(L > 0.0f) || !(b > 0.0f)) return ORACLE_ERR_ARG;
    int64_t n = (int64_t)floor((double)L / (double)b);
    if (n < 3) { *P_out = (uint64_t)N * (uint64_t)(N > 0 ? N - 1 : 0) / 2; return ORACLE_OK; }
    int64_t *key = (int64_t *)malloc(sizeof(int64_t) * (size_t)(N > 0 ? N : 1));
    int64_t *cnt = (int64_t *)malloc(sizeof(int64_t) * (size_t)(N > 0 ? N : 1));
    if (!key || !cnt) { free(key); free(cnt); return ORACLE_ERR_NOMEM; }
    double s = (double)n / (double)L;
    for (int64_t i = 0; i < N; ++i) {
        int64_t c3[3];
        for (int k = 0; k < 3; ++k) {
            if (!isfinite(pos[3 * i + k])) { free(key); free(cnt); return ORACLE_ERR_NONFINITE; }
            int64_t c = (int64_t)floor((double)oracle_wrap1(pos[3 * i + k], L) * s);
            if (c < 0) c = 0;
            if (c > n - 1) c = n - 1;
            c3[k] = c;
        }
        key[i] = c3[0] + n * (c3[1] + n * c3[2]);
    }
    qsort(key, (size_t)N, sizeof(int64_t), cmp_i64);
    int64_t U = 0;
    for (int64_t i = 0; i < N;) {
        int64_t j = i;
        while (j < N && key[j] == key[i]) ++j;
        key[U] = key[i]; cnt[U] = j - i; ++U;
        i = j;
    }
    uint64_t P = 0;
    for (int64_t u = 0; u < U; ++u) {
        int64_t c = key[u], cx = c % n, cy = (c / n) % n, cz = c / (n * n);
        P += (uint64_t)cnt[u] * (uint64_t)(cnt[u] - 1) / 2;
        for (int dz = -1; dz <= 1; ++dz)
        for (int dy = -1; dy <= 1; ++dy)
        for (int dx = -1; dx <= 1; ++dx) {
            if (dz < 0 || (dz == 0 && (dy < 0 || (dy == 0 && dx <= 0)))) continue;  /* 13 of 26 */
            int64_t m = (cx + dx + n) % n + n * ((cy + dy + n) % n + n * ((cz + dz + n) % n));
            P += (uint64_t)cnt[u] * (uint64_t)occ_of(key, cnt, U, m);
        }
    }
    *P_out = P;
    free(key); free(cnt);
    return ORACLE_OK;
}

/* Eq. 1: l_link = b (V/N)^(1/3), V = L^3; evaluated in double, rounded once. */
float oracle_linking_length(float b_frac, float L, int64_t N)
{
    return (float)((double)b_frac * (double)L / cbrt((double)N));
}
