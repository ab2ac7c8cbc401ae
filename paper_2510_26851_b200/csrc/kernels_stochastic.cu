// kernels_stochastic.cu — stochastic-edge Friends-of-Friends.
// PAPER.md section 3.2 (Eq. 6-8): every potential edge is y_ij ~ Bernoulli(p_ij),
// p_ij = sigma(alpha (b^2 - d_ij^2) / b^2); the halos of one Monte Carlo sample are the connected
// components of the sampled edges, and REINFORCE (Eq. 7) needs log p(y) and its gradient.
// Readings R25-R28 of DESIGN.md: potential edges = pairs within the candidate radius the plan was
// created with; sigma = the logistic evaluated by a fixed float32 recipe; counter-based randomness
// keyed on (seed, sample, original indices); d log p / d x_i = sum_j (y - p)(-2 alpha delta / b^2).
// The binning is NOT redone: the kernel walks the cell-sorted arrays that the last fof_link left in
// the workspace ("we do not rebuild the neighbor list", and S samples share one sort).
// One warp per 32 home particles (a tile); candidates staged in shared memory, potential edges flattened over the lanes.
#include "fof_internal.cuh"

namespace fof {

// R26: the fixed float32 logistic (same sequence of IEEE operations as the oracle, no FMA).
// Also returns e = 2^(-t log2 e) (t clamped), so that log p = -log1p(e) and log(1 - p) = log p - t.
__device__ __forceinline__ float sigmoid_fixed(float t, float &e_out)
{
    t = fminf(fmaxf(t, -30.0f), 30.0f);
    const float z = __fmul_rn(-t, 1.44269504088896340736f);
    const float n = rintf(z);
    const float f = __fsub_rn(z, n);
    float q = 1.5403530393381609954e-4f;
    q = __fadd_rn(__fmul_rn(q, f), 1.3333558146428443423e-3f);
    q = __fadd_rn(__fmul_rn(q, f), 9.6181291076284771619e-3f);
    q = __fadd_rn(__fmul_rn(q, f), 5.5504108664821579953e-2f);
    q = __fadd_rn(__fmul_rn(q, f), 2.4022650695910071233e-1f);
    q = __fadd_rn(__fmul_rn(q, f), 6.9314718055994530942e-1f);
    q = __fadd_rn(__fmul_rn(q, f), 1.0f);
    const float e = __fmul_rn(q, __int_as_float(((int)n + 127) << 23));  // exact: |n| <= 44
    e_out = e;
    return __frcp_rn(__fadd_rn(1.0f, e));  // correctly rounded 1 / x: the bits of the oracle's division
}

// R27: 24 random bits from (folded seed, sample, lo, hi): two rounds of a 32-bit finaliser.
__device__ __forceinline__ unsigned int mix32(unsigned int x)
{
    x ^= x >> 16; x *= 0x7FEB352DU;
    x ^= x >> 15; x *= 0x846CA68BU;
    x ^= x >> 16;
    return x;
}

__device__ __forceinline__ unsigned int rng_u24(unsigned int key, unsigned int lo, unsigned int hi)
{
    unsigned int h = mix32(key + lo);
    h = mix32(h ^ (hi * 0x85EBCA6BU));
    return h >> 8;
}

struct StochParams {
    float b2;          // fl(b_link * b_link): the scale of Eq. 8
    float c;           // fl(alpha / b2): t = c (b2 - d2)
    float gscale;      // -2 c
    unsigned int key;  // mix32(fold(seed) ^ (sample * 0x9E3779B9))
};

__global__ void __launch_bounds__(kBlock) iota_kernel(int *__restrict__ labels, int64_t N)
{
    const int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (i < N) labels[i] = (int)i;
}

constexpr int kStochWarps = kBlock / 32;

#ifndef FOF_STOCH_DIRECT
#define FOF_STOCH_DIRECT 16  // direct form when the mean number of edges per lane is at least FOF_STOCH_DIRECT / 32 of the largest
#endif
struct StochAcc {
    float lp;  // a lane adds at most a few thousand O(1) terms: float32 is enough before the float64 reduction
    unsigned int ncand, nedge;
    float gx, gy, gz;  // gradient terms of this lane's own home particle gathered by the direct form of stoch_batch
};

// One warp per 32 consecutive cell-sorted home particles.  Homes of
// one grid row (same cy, cz: consecutive lanes, their cells consecutive in x) form a segment; its
// candidates are the nine rows around it, each one contiguous run of `sorted` (cells xa - 1 .. xb + 1;
// the periodic images of the end cells as runs of their own).  Candidates that cannot be within the
// candidate radius of the segment (too far from the face(s) they share with it) are dropped, the
// rest are staged 32 at a time in shared memory and every home tests every candidate (broadcast
// reads, ~13 instructions per 32 tests).  The pairs that pass — the potential edges — are then
// flattened home by home over the lanes for the expensive part (logistic, random draw, log p,
// gradient, hook), so that this part runs with full lanes and a home particle's gradient terms are
// consecutive (segmented warp scan, no atomics, fixed summation order).  A pair is owned (counted,
// log p, hooked) by its member with the smaller cell-sorted slot; seen from the other side the same
// pair (same p, same y: the generator is keyed on the pair) only feeds the home particle's gradient.
struct StochSmem {
    float4 home[32];  // x, y, z, original index
    float4 cand[64];  // x, y, z, cell-sorted slot
    float g[32][3];
    int selfk[32];    // 1 + position in the batch of the home's own slot, 0 if it is not there
};

// Lane h: the candidates of the batch within the candidate radius of home h (bit k: candidate k).
template <bool WRAP>
__device__ __forceinline__ unsigned int stoch_adjacency(const float4 *cand, int cnt, const float4 &mine, const Grid &g)
{
    unsigned int adjH = 0;
#pragma unroll 4
    for (int k = 0; k < cnt; ++k) {
        const float4 pj = cand[k];
        float ddx = __fsub_rn(mine.x, pj.x), ddy = __fsub_rn(mine.y, pj.y), ddz = __fsub_rn(mine.z, pj.z);
        if (WRAP) {
            ddx = min_image(ddx, g.L, g.h);
            ddy = min_image(ddy, g.L, g.h);
            ddz = min_image(ddz, g.L, g.h);
        }
        const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(ddx, ddx), __fmul_rn(ddy, ddy)), __fmul_rn(ddz, ddz));
        if (d2 <= g.b2) adjH |= 1u << k;  // R25: beyond the radius p = 0
    }
    return adjH;
}

// position of the (r + 1)-th set bit of m (r < popc(m))
__device__ __forceinline__ int nth_set_bit(unsigned int m, int r)
{
    int pos = 0;
#pragma unroll
    for (int w = 16; w > 0; w >>= 1) {
        const int c = __popc(m & ((1u << w) - 1u));
        if (r >= c) { r -= c; pos += w; m >>= w; }
    }
    return pos;
}

// Every home against every candidate of the batch; a home's own slot is taken out afterwards.
__device__ __forceinline__ unsigned int stoch_batch_adjacency(StochSmem &sm, int cnt, bool wrap, const float4 &mine,
                                                              int s0, const Grid &g, int lane)
{
    sm.selfk[lane] = 0;
    __syncwarp();
    if (lane < cnt) {
        const unsigned int d = (unsigned int)(__float_as_int(sm.cand[lane].w) - s0);
        if (d < 32u) sm.selfk[d] = lane + 1;
    }
    unsigned int adjH = wrap ? stoch_adjacency<true>(sm.cand, cnt, mine, g) : stoch_adjacency<false>(sm.cand, cnt, mine, g);
    __syncwarp();
    const int sk = sm.selfk[lane];
    if (sk) adjH &= ~(1u << (sk - 1));
    return adjH;
}

__device__ __forceinline__ void stoch_batch(StochSmem &sm, int cnt, bool wrap, const float4 &mine, int myslot, int s0,
                                            const Grid &g, const StochParams &sp, const int *__restrict__ idx_s,
                                            unsigned int *rel, bool want_grad, int lane, StochAcc &acc)
{
    constexpr unsigned int kAll = 0xffffffffu;
    unsigned int adjH = stoch_batch_adjacency(sm, cnt, wrap, mine, s0, g, lane);
    // ---- the potential edges, home-major, 32 at a time
    const int mine_n = __popc(adjH);
    int incl = mine_n;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(kAll, incl, o);
        if (lane >= o) incl += v;
    }
    const int total = __shfl_sync(kAll, incl, 31);
    const int excl = incl - mine_n;
    if (__reduce_max_sync(kAll, mine_n) * FOF_STOCH_DIRECT <= total) {
        // Every home has about as many potential edges as the busiest one (a clump core): each lane walks
        // its own, no flattening, the gradient stays in registers.
        const float4 ph = sm.home[lane];
        unsigned int m = adjH;
        while (__any_sync(kAll, m != 0u)) {
            if (m) {
                const float4 pj = sm.cand[__ffs((int)m) - 1];
                m &= m - 1u;
                const int j = __float_as_int(pj.w);
                const bool owned = j > myslot;
                if (want_grad || owned) {
                    const float ddx = min_image(__fsub_rn(ph.x, pj.x), g.L, g.h);
                    const float ddy = min_image(__fsub_rn(ph.y, pj.y), g.L, g.h);
                    const float ddz = min_image(__fsub_rn(ph.z, pj.z), g.L, g.h);
                    const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(ddx, ddx), __fmul_rn(ddy, ddy)), __fmul_rn(ddz, ddz));
                    const float tt = __fmul_rn(sp.c, __fsub_rn(sp.b2, d2));
                    float e;
                    const float pr = sigmoid_fixed(tt, e);
                    const unsigned int ooi = (unsigned int)__float_as_int(ph.w), oj = (unsigned int)__ldg(idx_s + j);
                    const float u = __fmul_rn((float)rng_u24(sp.key, min(ooi, oj), max(ooi, oj)), 5.9604644775390625e-8f);
                    const bool y = u < pr;
                    const float tc = fminf(fmaxf(tt, -30.0f), 30.0f);
                    if (want_grad && tt == tc) {
                        const float cgr = ((y ? 1.0f : 0.0f) - pr) * sp.gscale;
                        acc.gx += cgr * ddx;
                        acc.gy += cgr * ddy;
                        acc.gz += cgr * ddz;
                    }
                    if (owned) {
                        ++acc.ncand;
                        acc.lp += -__logf(__fadd_rn(1.0f, e)) - (y ? 0.0f : tc);
                        if (y) {
                            ++acc.nedge;
                            const int pa = myslot - (int)rel[myslot], pb = j - (int)rel[j];
                            if (pa != pb) unite_rel(rel, idx_s, myslot, j);  // same parent: already one set
                        }
                    }
                }
            }
        }
        return;
    }
    for (int p0 = 0; p0 < total; p0 += 32) {
        const int p = p0 + lane;
        const bool has = p < total;
        int owner = 0;  // the first lane whose inclusive prefix exceeds p
#pragma unroll
        for (int st = 16; st > 0; st >>= 1) {
            const int v = __shfl_sync(kAll, incl, owner + st - 1);
            if (v <= p) owner += st;
        }
        owner = min(owner, 31);
        const unsigned int mask = __shfl_sync(kAll, adjH, owner);
        const int rank = p - __shfl_sync(kAll, excl, owner);
        const int osi = s0 + owner;
        float gx = 0.0f, gy = 0.0f, gz = 0.0f;
        if (has) {
            const float4 ph = sm.home[owner], pj = sm.cand[nth_set_bit(mask, rank)];
            const int j = __float_as_int(pj.w);
            // the owner of a pair: its member with the smaller cell-sorted slot
            const bool owned = j > osi;
            if (want_grad || owned) {  // without the gradient only the owning side has work
                const float ddx = min_image(__fsub_rn(ph.x, pj.x), g.L, g.h);
                const float ddy = min_image(__fsub_rn(ph.y, pj.y), g.L, g.h);
                const float ddz = min_image(__fsub_rn(ph.z, pj.z), g.L, g.h);
                const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(ddx, ddx), __fmul_rn(ddy, ddy)), __fmul_rn(ddz, ddz));
                const float tt = __fmul_rn(sp.c, __fsub_rn(sp.b2, d2));
                float e;
                const float pr = sigmoid_fixed(tt, e);
                const unsigned int ooi = (unsigned int)__float_as_int(ph.w), oj = (unsigned int)__ldg(idx_s + j);
                const float u = __fmul_rn((float)rng_u24(sp.key, min(ooi, oj), max(ooi, oj)), 5.9604644775390625e-8f);
                const bool y = u < pr;
                const float tc = fminf(fmaxf(tt, -30.0f), 30.0f);
                if (want_grad && tt == tc) {
                    const float cgr = ((y ? 1.0f : 0.0f) - pr) * sp.gscale;
                    gx = cgr * ddx;
                    gy = cgr * ddy;
                    gz = cgr * ddz;
                }
                if (owned) {
                    ++acc.ncand;
                    // log p = -log(1 + e); log(1 - p) = log(e / (1 + e)) = log p - t; float32 terms
                    acc.lp += -__logf(__fadd_rn(1.0f, e)) - (y ? 0.0f : tc);
                    if (y) {
                        ++acc.nedge;
                        const int pa = osi - (int)rel[osi], pb = j - (int)rel[j];
                        if (pa != pb) unite_rel(rel, idx_s, osi, j);  // same parent: already one set
                    }
                }
            }
        }
        if (want_grad && __any_sync(kAll, gx != 0.0f || gy != 0.0f || gz != 0.0f)) {
            // segmented inclusive scan over runs of equal owner, then one add per home particle
            const int key = has ? owner : -1 - lane;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const float vx = __shfl_up_sync(kAll, gx, o), vy = __shfl_up_sync(kAll, gy, o),
                            vz = __shfl_up_sync(kAll, gz, o);
                const int kk = __shfl_up_sync(kAll, key, o);
                if (lane >= o && kk == key) { gx += vx; gy += vy; gz += vz; }
            }
            const int knext = __shfl_down_sync(kAll, key, 1);
            if (has && (lane == 31 || knext != key)) {
                sm.g[owner][0] += gx;
                sm.g[owner][1] += gy;
                sm.g[owner][2] += gz;
            }
            __syncwarp();
        }
    }
}

// What happens to one staged batch: one sample (BatchOne) or several samples at once (BatchMulti).
struct BatchOne {
    const Grid &g;
    const StochParams &sp;
    const int *__restrict__ idx_s;
    unsigned int *rel;
    bool want_grad;
    StochAcc &acc;
    __device__ __forceinline__ void operator()(StochSmem &sm, int cnt, bool wrap, const float4 &mine, int myslot, int s0,
                                               int lane) const
    {
        stoch_batch(sm, cnt, wrap, mine, myslot, s0, g, sp, idx_s, rel, want_grad, lane, acc);
    }
};

// SB samples in one pass: candidate filter, distance tests and p_ij do not depend on the sample; only the
// draw, the log terms, the gradient terms and the hooks (one union-find array per sample) do.  Each
// lane walks the potential edges of its own home particle; all accumulators are registers.
template <int SB>
struct BatchMulti {
    const Grid &g;
    const StochParams &sp;
    const unsigned int *keys;  // per-sample generator keys
    const int *__restrict__ idx_s;
    unsigned int *rel;         // SB arrays of N
    int64_t N;
    bool want_grad;
    float *lp;                 // [SB]
    unsigned int *nedge;       // [SB]
    float (*gr)[3];            // [SB][3]
    unsigned int &ncand;
    __device__ __forceinline__ void operator()(StochSmem &sm, int cnt, bool wrap, const float4 &mine, int myslot, int s0,
                                               int lane) const
    {
        unsigned int m = stoch_batch_adjacency(sm, cnt, wrap, mine, s0, g, lane);
        const float4 ph = sm.home[lane];
        while (__any_sync(0xffffffffu, m != 0u)) {
            if (m) {
                const float4 pj = sm.cand[__ffs((int)m) - 1];
                m &= m - 1u;
                const int j = __float_as_int(pj.w);
                const bool owned = j > myslot;
                if (want_grad || owned) {
                    const float ddx = min_image(__fsub_rn(ph.x, pj.x), g.L, g.h);
                    const float ddy = min_image(__fsub_rn(ph.y, pj.y), g.L, g.h);
                    const float ddz = min_image(__fsub_rn(ph.z, pj.z), g.L, g.h);
                    const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(ddx, ddx), __fmul_rn(ddy, ddy)), __fmul_rn(ddz, ddz));
                    const float tt = __fmul_rn(sp.c, __fsub_rn(sp.b2, d2));
                    float e;
                    const float pr = sigmoid_fixed(tt, e);
                    const unsigned int ooi = (unsigned int)__float_as_int(ph.w), oj = (unsigned int)__ldg(idx_s + j);
                    const unsigned int klo = min(ooi, oj), khi = max(ooi, oj);
                    const float tc = fminf(fmaxf(tt, -30.0f), 30.0f);
                    const float lp1 = -__logf(__fadd_rn(1.0f, e));
                    const bool gon = want_grad && tt == tc;
                    if (owned) ++ncand;
#pragma unroll
                    for (int sidx = 0; sidx < SB; ++sidx) {
                        const float u = __fmul_rn((float)rng_u24(keys[sidx], klo, khi), 5.9604644775390625e-8f);
                        const bool y = u < pr;
                        if (gon) {
                            const float cgr = ((y ? 1.0f : 0.0f) - pr) * sp.gscale;
                            gr[sidx][0] += cgr * ddx;
                            gr[sidx][1] += cgr * ddy;
                            gr[sidx][2] += cgr * ddz;
                        }
                        if (owned) {
                            lp[sidx] += lp1 - (y ? 0.0f : tc);
                            if (y) {
                                ++nedge[sidx];
                                unsigned int *r = rel + (int64_t)sidx * N;
                                const int pa = myslot - (int)r[myslot], pb = j - (int)r[j];
                                if (pa != pb) unite_rel(r, idx_s, myslot, j);
                            }
                        }
                    }
                }
            }
        }
    }
};

template <class Batch>
__device__ __forceinline__ void stoch_tile_warp(const float4 *__restrict__ sorted, const Grid &g,
                                                const unsigned int *__restrict__ cs,
                                                StochSmem &sm, const float4 &me, int myslot, unsigned int oi,
                                                bool valid, int cx, int cy, int cz, int lane, const Batch &batch)
{
    constexpr unsigned int kAll = 0xffffffffu;
    const float inf = __int_as_float(0x7f800000);
    const int n = g.n;
    const int row = cy + n * cz;
    const int s0 = __shfl_sync(kAll, myslot, 0);  // slot of lane 0 (lanes past the end of the array repeat the last slot)
    const float lo = g.reach, hi = 1.0f - g.reach;
    sm.home[lane] = make_float4(me.x, me.y, me.z, __int_as_float((int)oi));
    __syncwarp();

    unsigned int todo = __ballot_sync(kAll, valid);
    while (todo) {
        const int l0 = __ffs((int)todo) - 1;
        const int r0 = __shfl_sync(kAll, row, l0);
        const unsigned int seg = __ballot_sync(kAll, valid && row == r0) & todo;
        todo &= ~seg;
        const bool inseg = (seg >> lane) & 1u;
        const int xa = __shfl_sync(kAll, cx, l0), xb = __shfl_sync(kAll, cx, 31 - __clz((int)seg));
        const int cy0 = __shfl_sync(kAll, cy, l0), cz0 = __shfl_sync(kAll, cz, l0);
        // a lane outside the segment sits at +inf: d2 = inf (or NaN) fails every test
        const float4 mine = inseg ? me : make_float4(inf, inf, inf, 0.0f);
        const int span = xb - xa + 1;
        const int xl = xa > 0 ? xa - 1 : n - 1, xr = xb < n - 1 ? xb + 1 : 0;  // the cells beside the segment
        const bool edges = span <= n - 2;  // otherwise the end cells are inside the segment or coincide
        // away from the box faces no pair of the segment needs the minimum image (cf. link_kernel)
        const bool wrap = n < 6 || xa == 0 || xb == n - 1 || cy0 == 0 || cy0 == n - 1 || cz0 == 0 || cz0 == n - 1;
        // candidate runs: lane q < 27 = 3 (row of the stencil) + part; part 0: cells max(xa - 1, 0) ..
        // min(xb + 1, n - 1), part 1: cell n - 1 as the left image, part 2: cell 0 as the right image
        int beg = 0, len = 0;
        if (lane < 27) {
            const int rq = lane / 3, part = lane - 3 * rq;
            const int dy = rq % 3 - 1, dz = rq / 3 - 1;
            int ay = cy0 + dy, az = cz0 + dz;
            ay = ay < 0 ? n - 1 : (ay >= n ? 0 : ay);
            az = az < 0 ? n - 1 : (az >= n ? 0 : az);
            const int m0 = max(xa - 1, 0), m1 = min(xb + 1, n - 1);
            int c0 = -1, c1 = -1;
            if (part == 0) { c0 = m0; c1 = m1; }
            else if (part == 1) { if (xa == 0 && m1 < n - 1) c0 = c1 = n - 1; }
            else { if (xb == n - 1 && m0 > 0) c0 = c1 = 0; }
            if (c0 >= 0) {
                beg = (int)__ldg(cs + cell_id(c0, ay, az, n));
                len = (int)__ldg(cs + cell_id(c1, ay, az, n) + 1) - beg;
            }
        }
        int incl = len;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(kAll, incl, o);
            if (lane >= o) incl += v;
        }
        const int total = __shfl_sync(kAll, incl, 31);
        const int excl = incl - len;
        int nc = 0;  // candidates waiting in sm.cand (warp-uniform)
        for (int base = 0;; base += 32) {
            if (base < total) {
                const int p = base + lane;
                const bool has = p < total;
                int q = 0;  // owner run of slot p: the first lane whose inclusive prefix exceeds p
#pragma unroll
                for (int st = 16; st > 0; st >>= 1) {
                    const int v = __shfl_sync(kAll, incl, q + st - 1);
                    if (v <= p) q += st;
                }
                q = min(q, 31);
                const int j = __shfl_sync(kAll, beg, q) + (p - __shfl_sync(kAll, excl, q));
                bool pass = false;
                float4 pj = make_float4(0.f, 0.f, 0.f, 0.f);
                if (has) {
                    pj = __ldg(sorted + j);
                    // position of the candidate inside ITS cell: it can reach the segment only from within
                    // `reach` of the face(s) between its cell and the segment's cells
                    const float ux = __fmul_rn(pj.x, g.inv_cell), uy = __fmul_rn(pj.y, g.inv_cell),
                                uz = __fmul_rn(pj.z, g.inv_cell);
                    const int jx = min(__float2int_rd(ux), g.n_minus_1);
                    const float fx = ux - (float)jx;
                    const float fy = uy - (float)min(__float2int_rd(uy), g.n_minus_1);
                    const float fz = uz - (float)min(__float2int_rd(uz), g.n_minus_1);
                    const int rq = q / 3;
                    const int dy = rq % 3 - 1, dz = rq / 3 - 1;
                    pass = (dy == 0 || (dy < 0 ? fy > hi : fy < lo)) && (dz == 0 || (dz < 0 ? fz > hi : fz < lo));
                    if (edges) {
                        if (jx == xl) pass = pass && fx > hi;
                        if (jx == xr) pass = pass && fx < lo;
                    }
                    pj.w = __int_as_float(j);
                }
                const unsigned int bal = __ballot_sync(kAll, pass);
                if (pass) sm.cand[nc + __popc(bal & ((1u << lane) - 1u))] = pj;
                nc += __popc(bal);
                __syncwarp();
            }
            const bool last = base + 32 >= total;
            if (nc >= 32 || (last && nc)) {
                const int cnt = min(nc, 32);
                batch(sm, cnt, wrap, mine, myslot, s0, lane);
                const float4 keep = sm.cand[32 + lane];
                __syncwarp();
                sm.cand[lane] = keep;
                nc -= cnt;
                __syncwarp();
            }
            if (last && nc == 0) break;
        }
    }
    __syncwarp();
}

#ifndef FOF_STOCH_MINB
#define FOF_STOCH_MINB 6  // resident CTAs per SM the kernel is compiled for (register cap 40)
#endif
__global__ void __launch_bounds__(kBlock, FOF_STOCH_MINB) link_stochastic_kernel(const float4 *__restrict__ sorted, int64_t N, Grid g,
                                                                 const unsigned int *__restrict__ cs,
                                                                 const int *__restrict__ idx_s, unsigned int *rel,
                                                                 StochParams sp, double *logp, float *grad,
                                                                 Ctrl *ctrl)
{
    constexpr unsigned int kAll = 0xffffffffu;
    __shared__ StochSmem s_all[kStochWarps];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    StochSmem &sm = s_all[wib];
    const int64_t s64 = ((int64_t)blockIdx.x * kStochWarps + wib) * 32 + lane;
    const bool valid = s64 < N;
    const int myslot = (int)min(s64, N - 1);
    const float4 me = __ldg(sorted + myslot);
    const unsigned int oi = (unsigned int)__ldg(idx_s + myslot);
    const int cx = min(__float2int_rd(__fmul_rn(me.x, g.inv_cell)), g.n_minus_1),
              cy = min(__float2int_rd(__fmul_rn(me.y, g.inv_cell)), g.n_minus_1),
              cz = min(__float2int_rd(__fmul_rn(me.z, g.inv_cell)), g.n_minus_1);
    const bool want_grad = grad != nullptr;
    StochAcc acc = {0.0f, 0u, 0u, 0.0f, 0.0f, 0.0f};
    sm.g[lane][0] = sm.g[lane][1] = sm.g[lane][2] = 0.0f;
    __syncwarp();
    const BatchOne batch = {g, sp, idx_s, rel, want_grad, acc};
    stoch_tile_warp(sorted, g, cs, sm, me, myslot, oi, valid, cx, cy, cz, lane, batch);
    __syncwarp();
    if (want_grad && valid) {
        grad[3 * (int64_t)oi + 0] = sm.g[lane][0] + acc.gx;
        grad[3 * (int64_t)oi + 1] = sm.g[lane][1] + acc.gy;
        grad[3 * (int64_t)oi + 2] = sm.g[lane][2] + acc.gz;
    }
    double lpd = (double)acc.lp;
    unsigned int ncand = acc.ncand, nedge = acc.nedge;
    for (int o = 16; o > 0; o >>= 1) {
        lpd += __shfl_xor_sync(kAll, lpd, o);
        ncand += __shfl_xor_sync(kAll, ncand, o);
        nedge += __shfl_xor_sync(kAll, nedge, o);
    }
    if (lane == 0) {
        if (lpd != 0.0) atomicAdd(logp, lpd);
        if (ncand) atomicAdd(&ctrl->pair_tests, (unsigned long long)ncand);  // potential edges of this sample
        if (nedge) atomicAdd(&ctrl->edges, (unsigned long long)nedge);       // sampled edges
    }
}

// SB samples of the same binning in one pass (fof_link_stochastic_batch).  keys: one generator key per
// sample; rel: SB union-find arrays of N; logp: SB doubles; grad: SB arrays of [N][3] or nullptr.
struct StochKeys {
    unsigned int k[4];
    int count_potential;  // the pass that reports the potential edges (they are the same in every pass)
};

template <int SB>
__global__ void __launch_bounds__(kBlock, 4) link_stochastic_multi_kernel(const float4 *__restrict__ sorted, int64_t N,
                                                                          Grid g, const unsigned int *__restrict__ cs,
                                                                          const int *__restrict__ idx_s,
                                                                          unsigned int *rel, StochParams sp,
                                                                          StochKeys keys, double *logp, float *grad,
                                                                          Ctrl *ctrl)
{
    constexpr unsigned int kAll = 0xffffffffu;
    __shared__ StochSmem s_all[kStochWarps];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    StochSmem &sm = s_all[wib];
    const int64_t s64 = ((int64_t)blockIdx.x * kStochWarps + wib) * 32 + lane;
    const bool valid = s64 < N;
    const int myslot = (int)min(s64, N - 1);
    const float4 me = __ldg(sorted + myslot);
    const unsigned int oi = (unsigned int)__ldg(idx_s + myslot);
    const int cx = min(__float2int_rd(__fmul_rn(me.x, g.inv_cell)), g.n_minus_1),
              cy = min(__float2int_rd(__fmul_rn(me.y, g.inv_cell)), g.n_minus_1),
              cz = min(__float2int_rd(__fmul_rn(me.z, g.inv_cell)), g.n_minus_1);
    float lp[SB], gr[SB][3];
    unsigned int nedge[SB], ncand = 0;
#pragma unroll
    for (int k = 0; k < SB; ++k) { lp[k] = 0.0f; nedge[k] = 0u; gr[k][0] = gr[k][1] = gr[k][2] = 0.0f; }
    const BatchMulti<SB> batch = {g, sp, keys.k, idx_s, rel, N, grad != nullptr, lp, nedge, gr, ncand};
    stoch_tile_warp(sorted, g, cs, sm, me, myslot, oi, valid, cx, cy, cz, lane, batch);
    __syncwarp();
    unsigned int nedge_all = 0;
#pragma unroll
    for (int k = 0; k < SB; ++k) {
        if (grad && valid) {
            float *gk = grad + (int64_t)k * 3 * N + 3 * (int64_t)oi;
            gk[0] = gr[k][0];
            gk[1] = gr[k][1];
            gk[2] = gr[k][2];
        }
        double lpd = (double)lp[k];
        for (int o = 16; o > 0; o >>= 1) lpd += __shfl_xor_sync(kAll, lpd, o);
        if (lane == 0 && lpd != 0.0) atomicAdd(logp + k, lpd);
        nedge_all += nedge[k];
    }
    for (int o = 16; o > 0; o >>= 1) {
        ncand += __shfl_xor_sync(kAll, ncand, o);
        nedge_all += __shfl_xor_sync(kAll, nedge_all, o);
    }
    if (lane == 0) {
        if (ncand && keys.count_potential) atomicAdd(&ctrl->pair_tests, (unsigned long long)ncand);  // potential edges
        if (nedge_all) atomicAdd(&ctrl->edges, (unsigned long long)nedge_all);  // sampled edges, all samples of the call
    }
}

// =============================================================================================
// The potential-edge list ("we do not rebuild the neighbor list"; section 3.2: the S samples of a
// REINFORCE step share the neighbour structure).  Which pairs are potential edges, their p_ij, t_ij and
// displacement do not depend on the sample: fof_stochastic_list_build writes them down once, home particle by home
// particle in cell-sorted slot order (every potential edge under both of its particles, so that a particle's
// score-function terms are its own records: no atomics, fixed summation order), and a sample is one coalesced stream
// over the list: draw, log term, gradient term, hook.  A record is two 16-byte halves in two arrays (recA = rec,
// recB = rec + records):
//   A: cand   original index of the other particle; bit 31: this side OWNS the pair (its cell-sorted slot is the
//             smaller one): it counts the edge, adds its log term and hooks
//      p      p_ij (the bits the single-sample kernel compares the draw with)
//      slot   cell-sorted slot of the other particle
//      home   cell-sorted slot of the home particle
//   B: dx, dy, dz  minimum-image displacement home - other, or 0 where t was clamped (no gradient there)
//      t      t_ij clamped to [-30, 30]: log p - log(1 - p)
// =============================================================================================
struct BatchCount {
    const Grid &g;
    unsigned int &count;
    __device__ __forceinline__ void operator()(StochSmem &sm, int cnt, bool wrap, const float4 &mine, int myslot, int s0,
                                               int lane) const
    {
        count += (unsigned int)__popc(stoch_batch_adjacency(sm, cnt, wrap, mine, s0, g, lane));
    }
};

struct BatchFill {
    const Grid &g;
    const StochParams &sp;
    const int *__restrict__ idx_s;
    uint4 *recA, *recB;
    unsigned int &wr;     // this lane's next record
    double &lp0;          // sum over the pairs this lane owns of log(1 - p) = log p - t: float32 log p and t as the
                          // sample kernels, their difference and the sum in float64 (the sample pass adds t back for
                          // every sampled edge: that cancellation must be exact)
    unsigned int &ncand;  // pairs this lane owns
    __device__ __forceinline__ void operator()(StochSmem &sm, int cnt, bool wrap, const float4 &mine, int myslot, int s0,
                                               int lane) const
    {
        unsigned int m = stoch_batch_adjacency(sm, cnt, wrap, mine, s0, g, lane);
        const float4 ph = sm.home[lane];
        while (__any_sync(0xffffffffu, m != 0u)) {
            if (m) {
                const float4 pj = sm.cand[__ffs((int)m) - 1];
                m &= m - 1u;
                const int j = __float_as_int(pj.w);
                const bool owned = j > myslot;
                const float ddx = min_image(__fsub_rn(ph.x, pj.x), g.L, g.h);
                const float ddy = min_image(__fsub_rn(ph.y, pj.y), g.L, g.h);
                const float ddz = min_image(__fsub_rn(ph.z, pj.z), g.L, g.h);
                const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(ddx, ddx), __fmul_rn(ddy, ddy)), __fmul_rn(ddz, ddz));
                const float tt = __fmul_rn(sp.c, __fsub_rn(sp.b2, d2));
                float e;
                const float pr = sigmoid_fixed(tt, e);
                const float tc = fminf(fmaxf(tt, -30.0f), 30.0f);
                const unsigned int oj = (unsigned int)__ldg(idx_s + j);
                if (owned) {
                    ++ncand;
                    lp0 += (double)(-__logf(__fadd_rn(1.0f, e))) - (double)tc;
                }
                const bool gon = tt == tc;
                uint4 a, b;
                a.x = oj | (owned ? 0x80000000u : 0u);
                a.y = (unsigned int)__float_as_int(pr);
                a.z = (unsigned int)j;
                a.w = (unsigned int)myslot;
                b.x = (unsigned int)__float_as_int(gon ? ddx : 0.0f);
                b.y = (unsigned int)__float_as_int(gon ? ddy : 0.0f);
                b.z = (unsigned int)__float_as_int(gon ? ddz : 0.0f);
                b.w = (unsigned int)__float_as_int(tc);
                __stcs(recA + wr, a);
                __stcs(recB + wr, b);
                ++wr;
            }
        }
    }
};

// FILL = false: counts[slot] = number of records of the home particle in `slot`;
// FILL = true: the records, from roff[slot] on (the scanned counts), and home_orig[slot] = its original index.
template <bool FILL>
__global__ void __launch_bounds__(kBlock, FOF_STOCH_MINB) stoch_list_kernel(const float4 *__restrict__ sorted, int64_t N, Grid g,
                                                            const unsigned int *__restrict__ cs,
                                                            const int *__restrict__ idx_s, StochParams sp,
                                                            StochList list, unsigned int *counts)
{
    constexpr unsigned int kAll = 0xffffffffu;
    __shared__ StochSmem s_all[kStochWarps];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    StochSmem &sm = s_all[wib];
    const int64_t s64 = ((int64_t)blockIdx.x * kStochWarps + wib) * 32 + lane;
    const bool valid = s64 < N;
    const int myslot = (int)min(s64, N - 1);
    const float4 me = __ldg(sorted + myslot);
    const unsigned int oi = (unsigned int)__ldg(idx_s + myslot);
    const int cx = min(__float2int_rd(__fmul_rn(me.x, g.inv_cell)), g.n_minus_1),
              cy = min(__float2int_rd(__fmul_rn(me.y, g.inv_cell)), g.n_minus_1),
              cz = min(__float2int_rd(__fmul_rn(me.z, g.inv_cell)), g.n_minus_1);
    if (!FILL) {
        unsigned int count = 0;
        const BatchCount batch = {g, count};
        stoch_tile_warp(sorted, g, cs, sm, me, myslot, oi, valid, cx, cy, cz, lane, batch);
        if (valid) counts[myslot] = count;
    } else {
        if (valid) list.home_orig[myslot] = (int)oi;
        unsigned int wr = valid ? list.roff[myslot] : 0u, ncand = 0;
        double lp0 = 0.0;
        const BatchFill batch = {g, sp, idx_s, list.rec, list.rec + list.roff[N], wr, lp0, ncand};
        stoch_tile_warp(sorted, g, cs, sm, me, myslot, oi, valid, cx, cy, cz, lane, batch);
        __syncwarp();
        double lpd = lp0;
        for (int o = 16; o > 0; o >>= 1) {
            lpd += __shfl_xor_sync(kAll, lpd, o);
            ncand += __shfl_xor_sync(kAll, ncand, o);
        }
        if (lane == 0 && ncand) {
            atomicAdd(&list.head->logp0, lpd);
            atomicAdd(&list.head->potential, (unsigned long long)ncand);
        }
    }
}

// ---- exclusive scan of roff[0 .. N) in place, roff[N] = total (three small kernels: tile sums, their scan, apply)
constexpr int kListScanThreads = 512, kListScanPer = kListScanTile / kListScanThreads;

__device__ __forceinline__ unsigned long long block_exclusive_u64(unsigned long long v, unsigned long long *s_w,
                                                                  unsigned long long &total)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    unsigned long long incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    __syncthreads();  // s_w may still be read from a previous call
    if (lane == 31) s_w[w] = incl;
    __syncthreads();
    unsigned long long before = 0, all = 0;
    for (int k = 0; k < nw; ++k) {
        const unsigned long long t = s_w[k];
        if (k < w) before += t;
        all += t;
    }
    total = all;
    return before + incl - v;
}

__global__ void __launch_bounds__(kListScanThreads) list_scan_sums_kernel(const unsigned int *__restrict__ v, int64_t n,
                                                                          unsigned long long *bsum)
{
    __shared__ unsigned long long s_w[kListScanThreads / 32];
    const int64_t i0 = (int64_t)blockIdx.x * kListScanTile + (int64_t)threadIdx.x * kListScanPer;
    unsigned long long sum = 0;
#pragma unroll
    for (int k = 0; k < kListScanPer; ++k)
        if (i0 + k < n) sum += v[i0 + k];
    unsigned long long total;
    (void)block_exclusive_u64(sum, s_w, total);
    if (threadIdx.x == 0) bsum[blockIdx.x] = total;
}

__global__ void __launch_bounds__(1024) list_scan_top_kernel(unsigned long long *bsum, int nb, StochListHead *head)
{
    __shared__ unsigned long long s_w[32];
    unsigned long long carry = 0;
    for (int base = 0; base < nb; base += 1024) {
        const int i = base + (int)threadIdx.x;
        const unsigned long long v = i < nb ? bsum[i] : 0ull;
        unsigned long long total;
        const unsigned long long ex = block_exclusive_u64(v, s_w, total);
        if (i < nb) bsum[i] = carry + ex;
        carry += total;
    }
    if (threadIdx.x == 0) {
        head->records = carry;
        head->potential = 0ull;
        head->logp0 = 0.0;
    }
}

__global__ void __launch_bounds__(kListScanThreads) list_scan_apply_kernel(unsigned int *v, int64_t n,
                                                                           const unsigned long long *__restrict__ bsum,
                                                                           const StochListHead *head)
{
    __shared__ unsigned long long s_w[kListScanThreads / 32];
    const int64_t i0 = (int64_t)blockIdx.x * kListScanTile + (int64_t)threadIdx.x * kListScanPer;
    unsigned int x[kListScanPer];
    unsigned long long sum = 0;
#pragma unroll
    for (int k = 0; k < kListScanPer; ++k) {
        x[k] = i0 + k < n ? v[i0 + k] : 0u;
        sum += x[k];
    }
    unsigned long long total;
    unsigned long long run = bsum[blockIdx.x] + block_exclusive_u64(sum, s_w, total);
#pragma unroll
    for (int k = 0; k < kListScanPer; ++k) {
        if (i0 + k < n) v[i0 + k] = (unsigned int)run;
        run += x[k];
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) v[n] = (unsigned int)head->records;
}

// SB samples over the list.  One warp per 32 consecutive home particles = one contiguous run of records, read 32 at
// a time (coalesced 128-bit loads), every lane one record.  The gradient terms of a home particle are consecutive
// lanes: a segmented warp scan sums them (the segment structure is shared by the SB samples), a run that continues
// in the next 32 records is carried over in registers, and the lane that holds a particle's last record stores its
// total: every particle's sum is formed by this warp alone, in record order.
// The union-find of sample k is rel + k N, in cell-sorted slot space as in fof_link (neighbours in space are
// neighbours in memory), ordered by list.home_orig, which is idx_s.
#ifndef FOF_STREAM_BLOCK
#define FOF_STREAM_BLOCK 64   // small CTAs: the runs of neighbouring tiles differ a lot in length (a halo next to background)
#endif
#ifndef FOF_STREAM_MINB
#define FOF_STREAM_MINB 16
#endif
#ifndef FOF_STREAM_WAVES
#define FOF_STREAM_WAVES 8    // CTAs launched = SMs x resident CTAs per SM x this (cfg2: 1.79 / 1.82 / 1.68 ms per sample at 1 / 2 / 8; one CTA per two tiles: 1.83)
#endif
constexpr int kStreamBlock = FOF_STREAM_BLOCK;
template <int SB>
__global__ void __launch_bounds__(kStreamBlock, FOF_STREAM_MINB) stoch_stream_kernel(StochList list, int64_t N, StochKeys keys, float gscale,
                                                              unsigned int *rel, double *logp, float *grad, Ctrl *ctrl)
{
    constexpr unsigned int kAll = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const uint4 *__restrict__ recA = list.rec;
    const uint4 *__restrict__ recB = list.rec + list.roff[N];
    const bool want_grad = grad != nullptr;
    double lp[SB];  // sum of t over the sampled edges: cancels against the t inside list.head->logp0, hence float64
    float carry[SB][3];
    unsigned int nedge[SB];
#pragma unroll
    for (int k = 0; k < SB; ++k) { lp[k] = 0.0; nedge[k] = 0u; carry[k][0] = carry[k][1] = carry[k][2] = 0.0f; }
    // Tiles of 32 homes, dealt round-robin to the warps of a grid of a few waves: a halo's tiles hold hundreds of
    // records each, the field's a handful, and neighbouring tiles are alike: the deal evens that out without a ticket.
    const int64_t ntiles = (N + 31) >> 5;
    const int64_t nwarps = ((int64_t)gridDim.x * kStreamBlock) >> 5;
    for (int64_t tile = ((int64_t)blockIdx.x * kStreamBlock + threadIdx.x) >> 5; tile < ntiles; tile += nwarps) {
    const int64_t h0 = tile * 32;
    const unsigned int rb = list.roff[h0], re = list.roff[min(h0 + 32, N)];
    if (rb == re) continue;
    const unsigned int tile_orig = (unsigned int)__ldg(list.home_orig + min(h0 + lane, N - 1));  // lane l: original index of home h0 + l
    int prev_home = -1;  // home of the record before this batch
    // the next batch is loaded while this one is worked on
    uint4 an = make_uint4(0u, 0u, 0u, 0u), bn = make_uint4(0u, 0u, 0u, 0u);
    if (rb + lane < re) {
        an = __ldcs(recA + rb + lane);
        bn = __ldcs(recB + rb + lane);
    }
    for (unsigned int r0 = rb; r0 < re; r0 += 32) {
        const unsigned int r = r0 + lane;
        const bool has = r < re;
        const uint4 a = an, b = bn;
        an = make_uint4(0u, 0u, 0u, 0u);
        if (r + 32 < re) {
            an = __ldcs(recA + r + 32);
            bn = __ldcs(recB + r + 32);
        }
        const int home = has ? (int)a.w : -2 - lane;
        const bool owned = (a.x >> 31) != 0u;
        const unsigned int oj = a.x & 0x7fffffffu;
        const float pr = __int_as_float((int)a.y), tc = __int_as_float((int)b.w);
        const float ddx = __int_as_float((int)b.x), ddy = __int_as_float((int)b.y), ddz = __int_as_float((int)b.z);
        const int j = (int)a.z;
        const unsigned int ooi = __shfl_sync(kAll, tile_orig, (int)a.w - (int)h0);  // every home of the run is in my tile
        const unsigned int klo = min(ooi, oj), khi = max(ooi, oj);
        // segments of equal home: `first` = lane of my segment's first record in this batch; the last record of a
        // particle is where the next record (the next batch's first one for lane 31) has another home
        const int left = __shfl_up_sync(kAll, home, 1);
        const unsigned int heads = __ballot_sync(kAll, lane == 0 || left != home);
        const int first = 31 - __clz((int)(heads & (0xffffffffu >> (31 - lane))));
        int right = __shfl_down_sync(kAll, home, 1);
        const int next0 = __shfl_sync(kAll, (int)an.w, 0);  // home of the next batch's first record
        if (lane == 31) right = (r + 1 < re) ? next0 : -1;
        const bool tail = has && right != home;
        const bool cont = lane == first && first == 0 && home == prev_home;  // lane 0 continues the previous batch's run
        prev_home = __shfl_sync(kAll, home, 31);
        bool hook[SB];
#pragma unroll
        for (int k = 0; k < SB; ++k) {
            const float u = __fmul_rn((float)rng_u24(keys.k[k], klo, khi), 5.9604644775390625e-8f);
            const bool y = has && u < pr;
            hook[k] = owned && y;
            if (want_grad) {
                const float cgr = ((y ? 1.0f : 0.0f) - pr) * gscale;
                float gx = cgr * ddx, gy = cgr * ddy, gz = cgr * ddz;
                if (cont) { gx += carry[k][0]; gy += carry[k][1]; gz += carry[k][2]; }
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const float vx = __shfl_up_sync(kAll, gx, o), vy = __shfl_up_sync(kAll, gy, o),
                                vz = __shfl_up_sync(kAll, gz, o);
                    if (lane - o >= first) { gx += vx; gy += vy; gz += vz; }
                }
                if (tail) {
                    float *gk = grad + (int64_t)k * 3 * N + 3 * (int64_t)ooi;
                    gk[0] = gx;
                    gk[1] = gy;
                    gk[2] = gz;
                }
                carry[k][0] = __shfl_sync(kAll, gx, 31);
                carry[k][1] = __shfl_sync(kAll, gy, 31);
                carry[k][2] = __shfl_sync(kAll, gz, 31);
            }
            if (hook[k]) {
                lp[k] += (double)tc;
                ++nedge[k];
            }
        }
        // the hooks of the SB samples: first every parent load (independent, all in flight together), then the
        // unions that are not already inside one set
        int pa[SB], pb[SB];
#pragma unroll
        for (int k = 0; k < SB; ++k) {
            const unsigned int *rk = rel + (int64_t)k * N;
            pa[k] = pb[k] = 0;
            if (hook[k]) {
                pa[k] = home - (int)rk[home];
                pb[k] = j - (int)rk[j];
            }
        }
#pragma unroll
        for (int k = 0; k < SB; ++k)
            if (pa[k] != pb[k]) unite_rel(rel + (int64_t)k * N, list.home_orig, home, j);  // same parent: one set
    }
    }  // tiles
    const bool first_warp = blockIdx.x == 0 && threadIdx.x < 32;
    unsigned int nedge_all = 0;
#pragma unroll
    for (int k = 0; k < SB; ++k) {
        double lpd = lp[k];
        for (int o = 16; o > 0; o >>= 1) lpd += __shfl_xor_sync(kAll, lpd, o);
        if (first_warp) lpd += list.head->logp0;  // log p(y) = log p(all absent) + sum over the sampled edges of t
        if (lane == 0 && lpd != 0.0) atomicAdd(logp + k, lpd);
        nedge_all += nedge[k];
    }
    for (int o = 16; o > 0; o >>= 1) nedge_all += __shfl_xor_sync(kAll, nedge_all, o);
    if (lane == 0 && nedge_all) atomicAdd(&ctrl->edges, (unsigned long long)nedge_all);  // sampled edges, all samples
    if (first_warp && lane == 0 && keys.count_potential) ctrl->pair_tests = list.head->potential;
}

static inline unsigned int blocks_for(int64_t n, int per_block) { return (unsigned int)((n + per_block - 1) / per_block); }

static unsigned int stoch_key(unsigned long long seed, unsigned int sample)
{
    unsigned int k = (unsigned int)(seed ^ (seed >> 32)) ^ (sample * 0x9E3779B9U);  // per-sample key: mix32 on the host
    k ^= k >> 16; k *= 0x7FEB352DU;
    k ^= k >> 15; k *= 0x846CA68BU;
    k ^= k >> 16;
    return k;
}

cudaError_t launch_link_stochastic(const float4 *sorted, int64_t N, Grid g, const unsigned int *cell_start,
                                   const int *idx_s, unsigned int *rel, float b_link, float alpha,
                                   unsigned long long seed, unsigned int sample, int *labels, double *logp, float *grad,
                                   Ctrl *ctrl, cudaStream_t s)
{
    cudaError_t e;
    if ((e = cudaMemsetAsync(logp, 0, sizeof(double), s)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(&ctrl->edges, 0, 2 * sizeof(unsigned long long), s)) != cudaSuccess) return e;
    if (N <= 0) return cudaSuccess;
    if ((e = cudaMemsetAsync(rel, 0, (size_t)N * sizeof(unsigned int), s)) != cudaSuccess) return e;
    StochParams sp;
    sp.b2 = b_link * b_link;
    sp.c = alpha / sp.b2;
    sp.gscale = -2.0f * sp.c;
    sp.key = stoch_key(seed, sample);
    iota_kernel<<<blocks_for(N, kBlock), kBlock, 0, s>>>(labels, N);
    link_stochastic_kernel<<<blocks_for(N, kBlock), kBlock, 0, s>>>(sorted, N, g, cell_start, idx_s, rel, sp, logp, grad,
                                                                    ctrl);
    return launch_write_labels(rel, idx_s, labels, N, nullptr, nullptr, nullptr, 0, nullptr, s);
}

// S samples sample0 .. sample0 + S - 1 on one binning, four per pass (then one by one).
cudaError_t launch_link_stochastic_batch(const float4 *sorted, int64_t N, Grid g, const unsigned int *cell_start,
                                         const int *idx_s, unsigned int *rel_s, float b_link, float alpha,
                                         unsigned long long seed, unsigned int sample0, int S, int *labels,
                                         double *logp, float *grad, Ctrl *ctrl, cudaStream_t s)
{
    cudaError_t e;
    if ((e = cudaMemsetAsync(logp, 0, (size_t)S * sizeof(double), s)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(&ctrl->edges, 0, 2 * sizeof(unsigned long long), s)) != cudaSuccess) return e;
    if (N <= 0) return cudaSuccess;
    if ((e = cudaMemsetAsync(rel_s, 0, (size_t)S * (size_t)N * sizeof(unsigned int), s)) != cudaSuccess) return e;
    StochParams sp;
    sp.b2 = b_link * b_link;
    sp.c = alpha / sp.b2;
    sp.gscale = -2.0f * sp.c;
    sp.key = 0u;
    const unsigned int grid = blocks_for(N, kBlock);
    for (int k0 = 0; k0 < S;) {
        StochKeys keys = {{0u, 0u, 0u, 0u}, k0 == 0 ? 1 : 0};
        const int sb = S - k0 >= 4 ? 4 : 1;
        for (int k = 0; k < sb; ++k) keys.k[k] = stoch_key(seed, sample0 + (unsigned int)(k0 + k));
        unsigned int *rel = rel_s + (size_t)k0 * (size_t)N;
        float *gk = grad ? grad + (size_t)k0 * 3 * (size_t)N : nullptr;
        if (sb == 4)
            link_stochastic_multi_kernel<4><<<grid, kBlock, 0, s>>>(sorted, N, g, cell_start, idx_s, rel, sp, keys,
                                                                    logp + k0, gk, ctrl);
        else
            link_stochastic_multi_kernel<1><<<grid, kBlock, 0, s>>>(sorted, N, g, cell_start, idx_s, rel, sp, keys,
                                                                    logp + k0, gk, ctrl);
        k0 += sb;
    }
    for (int k = 0; k < S; ++k) {
        int *lab = labels + (size_t)k * (size_t)N;
        iota_kernel<<<grid, kBlock, 0, s>>>(lab, N);
        if ((e = launch_write_labels(rel_s + (size_t)k * (size_t)N, idx_s, lab, N, nullptr, nullptr, nullptr, 0, nullptr, s)) != cudaSuccess) return e;
    }
    return cudaGetLastError();
}

static StochParams stoch_params(float b_link, float alpha)
{
    StochParams sp;
    sp.b2 = b_link * b_link;
    sp.c = alpha / sp.b2;
    sp.gscale = -2.0f * sp.c;
    sp.key = 0u;
    return sp;
}

// counts[slot] = records of the home particle in `slot` (the neighbour search without the per-pair work)
cudaError_t launch_stoch_list_count(const float4 *sorted, int64_t N, Grid g, const unsigned int *cell_start,
                                    const int *idx_s, unsigned int *counts, cudaStream_t s)
{
    if (N <= 0) return cudaSuccess;
    StochList none = {};
    stoch_list_kernel<false><<<blocks_for(N, kBlock), kBlock, 0, s>>>(sorted, N, g, cell_start, idx_s,
                                                                      stoch_params(1.0f, 0.0f), none, counts);
    return cudaGetLastError();
}

// counts -> list.roff (exclusive scan, roff[N] = total) and list.head->records
cudaError_t launch_stoch_list_offsets(const unsigned int *counts, int64_t N, StochList list, cudaStream_t s)
{
    const int nb = (int)((N + kListScanTile) / kListScanTile);  // tiles over N + 1 entries
    cudaError_t e;
    if (N > 0 && (e = cudaMemcpyAsync(list.roff, counts, (size_t)N * sizeof(unsigned int), cudaMemcpyDeviceToDevice, s)) != cudaSuccess)
        return e;
    list_scan_sums_kernel<<<nb, kListScanThreads, 0, s>>>(list.roff, N, list.bsum);
    list_scan_top_kernel<<<1, 1024, 0, s>>>(list.bsum, nb, list.head);
    list_scan_apply_kernel<<<nb, kListScanThreads, 0, s>>>(list.roff, N, list.bsum, list.head);
    return cudaGetLastError();
}

cudaError_t launch_stoch_list_fill(const float4 *sorted, int64_t N, Grid g, const unsigned int *cell_start,
                                   const int *idx_s, float b_link, float alpha, StochList list, cudaStream_t s)
{
    if (N <= 0) return cudaSuccess;
    stoch_list_kernel<true><<<blocks_for(N, kBlock), kBlock, 0, s>>>(sorted, N, g, cell_start, idx_s,
                                                                     stoch_params(b_link, alpha), list, nullptr);
    return cudaGetLastError();
}

// S samples sample0 .. sample0 + S - 1 over the list, four per pass (then one by one).
cudaError_t launch_link_stochastic_list(StochList list, int64_t N, float b_link, float alpha, unsigned long long seed,
                                        unsigned int sample0, int S, unsigned int *rel_s, int *labels, double *logp,
                                        float *grad, Ctrl *ctrl, int num_sms, cudaStream_t s)
{
    cudaError_t e;
    if ((e = cudaMemsetAsync(logp, 0, (size_t)S * sizeof(double), s)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(&ctrl->edges, 0, 2 * sizeof(unsigned long long), s)) != cudaSuccess) return e;
    if (N <= 0) return cudaSuccess;
    if ((e = cudaMemsetAsync(rel_s, 0, (size_t)S * (size_t)N * sizeof(unsigned int), s)) != cudaSuccess) return e;
    // a particle without potential edges has no record: its score function is the zero written here
    if (grad && (e = cudaMemsetAsync(grad, 0, (size_t)S * (size_t)N * 3 * sizeof(float), s)) != cudaSuccess) return e;
    const StochParams sp = stoch_params(b_link, alpha);
    const unsigned int grid = blocks_for(N, kBlock);
    for (int k0 = 0; k0 < S;) {
        StochKeys keys = {{0u, 0u, 0u, 0u}, k0 == 0 ? 1 : 0};
        const int sb = S - k0 >= 4 ? 4 : 1;  // eight per pass: 96+ registers, 2.6 ms per sample instead of 1.8 at cfg2
        for (int k = 0; k < sb; ++k) keys.k[k] = stoch_key(seed, sample0 + (unsigned int)(k0 + k));
        unsigned int *rel = rel_s + (size_t)k0 * (size_t)N;
        float *gk = grad ? grad + (size_t)k0 * 3 * (size_t)N : nullptr;
        const unsigned int sgrid = (unsigned int)min((int64_t)blocks_for(N, kStreamBlock),
                                                     (int64_t)(num_sms > 0 ? num_sms : 148) * FOF_STREAM_MINB * FOF_STREAM_WAVES);
        if (sb == 4) stoch_stream_kernel<4><<<sgrid, kStreamBlock, 0, s>>>(list, N, keys, sp.gscale, rel, logp + k0, gk, ctrl);
        else stoch_stream_kernel<1><<<sgrid, kStreamBlock, 0, s>>>(list, N, keys, sp.gscale, rel, logp + k0, gk, ctrl);
        k0 += sb;
    }
    for (int k = 0; k < S; ++k) {
        int *lab = labels + (size_t)k * (size_t)N;
        iota_kernel<<<grid, kBlock, 0, s>>>(lab, N);
        if ((e = launch_write_labels(rel_s + (size_t)k * (size_t)N, list.home_orig, lab, N, nullptr, nullptr, nullptr, 0,
                                     nullptr, s)) != cudaSuccess) return e;
    }
    return cudaGetLastError();
}

}  // namespace fof
