// kernels_stochastic.cu — stochastic-edge Friends-of-Friends.
// PAPER.md section 3.2 (Eq. 6-8): every potential edge is y_ij ~ Bernoulli(p_ij),
// p_ij = sigma(alpha (b^2 - d_ij^2) / b^2); the halos of one Monte Carlo sample are the connected
// components of the sampled edges, and REINFORCE (Eq. 7) needs log p(y) and its gradient.
// Readings R25-R28 of DESIGN.md: potential edges = pairs within the candidate radius the plan was
// created with; sigma = the logistic evaluated by a fixed float32 recipe; counter-based randomness
// keyed on (seed, sample, original indices); d log p / d x_i = sum_j (y - p)(-2 alpha delta / b^2).
// The binning is NOT redone: the kernel walks the cell-sorted arrays that the last fof_link left in
// the workspace ("we do not rebuild the neighbor list", and S samples share one sort).
// First correct path: one thread per home particle, half stencil, reach filter, direct loops.
#include "fof_internal.cuh"

namespace fof {

// R26: the fixed float32 logistic (same sequence of IEEE operations as the oracle, no FMA).
__device__ __forceinline__ float sigmoid_fixed(float t)
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
    return __fdiv_rn(1.0f, __fadd_rn(1.0f, e));
}

// R27: 24 random bits from (seed, sample, lo, hi), two rounds of the splitmix64 finaliser.
__device__ __forceinline__ unsigned long long splitmix_fin(unsigned long long z)
{
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ULL;
    z ^= z >> 27; z *= 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return z;
}

__device__ __forceinline__ unsigned int rng_u24(unsigned long long seed, unsigned int sample, unsigned int lo,
                                                unsigned int hi)
{
    unsigned long long x = seed ^ (0x9E3779B97F4A7C15ULL * ((unsigned long long)sample + 1ULL));
    x = splitmix_fin(x + (unsigned long long)lo);
    x = splitmix_fin(x ^ ((unsigned long long)hi * 0xD1B54A32D192ED03ULL));
    return (unsigned int)(x >> 40);
}

struct StochParams {
    float b2;       // fl(b_link * b_link): the scale of Eq. 8
    float alpha;
    double gscale;  // -2 alpha / b2
    unsigned long long seed;
    unsigned int sample;
};

__global__ void __launch_bounds__(kBlock) iota_kernel(int *__restrict__ labels, int64_t N)
{
    const int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (i < N) labels[i] = (int)i;
}

// One home particle per thread: the rest of its cell, then the 13 forward cells it can reach.
__global__ void __launch_bounds__(kBlock) link_stochastic_kernel(const float4 *__restrict__ sorted, int64_t N, Grid g,
                                                                 const unsigned int *__restrict__ cs,
                                                                 const int *__restrict__ idx_s, unsigned int *rel,
                                                                 StochParams sp, double *logp, float *grad,
                                                                 Ctrl *ctrl)
{
    const int64_t s64 = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    double lp = 0.0;
    unsigned int ncand = 0, nedge = 0;
    if (s64 < N) {
        const int si = (int)s64;
        const float4 me = __ldg(sorted + si);
        const unsigned int oi = (unsigned int)__ldg(idx_s + si);
        const int n = g.n;
        const float ux = __fmul_rn(me.x, g.inv_cell), uy = __fmul_rn(me.y, g.inv_cell), uz = __fmul_rn(me.z, g.inv_cell);
        const int cx = min(__float2int_rd(ux), g.n_minus_1), cy = min(__float2int_rd(uy), g.n_minus_1),
                  cz = min(__float2int_rd(uz), g.n_minus_1);
        const float fx = ux - (float)cx, fy = uy - (float)cy, fz = uz - (float)cz;
        const float lo = g.reach, hi = 1.0f - g.reach;
        float gx = 0.0f, gy = 0.0f, gz = 0.0f;
        for (int q = 0; q < 14; ++q) {  // own cell, +x, rows (+1,0), (-1,+1), (0,+1), (+1,+1)
            const int dx = q == 0 ? 0 : (q == 1 ? 1 : (q - 2) % 3 - 1);
            const int dy = q < 2 ? 0 : (q < 5 ? 1 : (q < 8 ? -1 : (q < 11 ? 0 : 1)));
            const int dz = q < 5 ? 0 : 1;
            if ((dx < 0 && !(fx < lo)) || (dx > 0 && !(fx > hi)) || (dy < 0 && !(fy < lo)) || (dy > 0 && !(fy > hi)) ||
                (dz > 0 && !(fz > hi)))
                continue;
            int ax = cx + dx, ay = cy + dy, az = cz + dz;
            ax = ax < 0 ? n - 1 : (ax >= n ? 0 : ax);
            ay = ay < 0 ? n - 1 : (ay >= n ? 0 : ay);
            az = az >= n ? 0 : az;
            const unsigned int c = cell_id(ax, ay, az, n);
            const int beg = q == 0 ? si + 1 : (int)__ldg(cs + c), end = (int)__ldg(cs + c + 1);
            for (int t = beg; t < end; ++t) {
                const float4 pj = __ldg(sorted + t);
                const float ddx = min_image(__fsub_rn(me.x, pj.x), g.L, g.h);
                const float ddy = min_image(__fsub_rn(me.y, pj.y), g.L, g.h);
                const float ddz = min_image(__fsub_rn(me.z, pj.z), g.L, g.h);
                const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(ddx, ddx), __fmul_rn(ddy, ddy)), __fmul_rn(ddz, ddz));
                if (!(d2 <= g.b2)) continue;  // R25: beyond the candidate radius p = 0
                ++ncand;
                const float tt = __fmul_rn(sp.alpha, __fdiv_rn(__fsub_rn(sp.b2, d2), sp.b2));
                const float p = sigmoid_fixed(tt);
                const unsigned int oj = (unsigned int)__ldg(idx_s + t);
                const float u = __fmul_rn((float)rng_u24(sp.seed, sp.sample, min(oi, oj), max(oi, oj)),
                                          5.9604644775390625e-8f);
                const bool y = u < p;
                lp += y ? log((double)p) : log1p(-(double)p);
                if (grad && tt <= 30.0f && tt >= -30.0f) {
                    const float cgr = (float)(((y ? 1.0 : 0.0) - (double)p) * sp.gscale);
                    const float ax_ = cgr * ddx, ay_ = cgr * ddy, az_ = cgr * ddz;
                    gx += ax_; gy += ay_; gz += az_;
                    atomicAdd(grad + 3 * (int64_t)oj + 0, -ax_);
                    atomicAdd(grad + 3 * (int64_t)oj + 1, -ay_);
                    atomicAdd(grad + 3 * (int64_t)oj + 2, -az_);
                }
                if (y) {
                    ++nedge;
                    unite_rel(rel, idx_s, si, t);
                }
            }
        }
        if (grad && (gx != 0.0f || gy != 0.0f || gz != 0.0f)) {
            atomicAdd(grad + 3 * (int64_t)oi + 0, gx);
            atomicAdd(grad + 3 * (int64_t)oi + 1, gy);
            atomicAdd(grad + 3 * (int64_t)oi + 2, gz);
        }
    }
    for (int o = 16; o > 0; o >>= 1) {
        lp += __shfl_xor_sync(0xffffffffu, lp, o);
        ncand += __shfl_xor_sync(0xffffffffu, ncand, o);
        nedge += __shfl_xor_sync(0xffffffffu, nedge, o);
    }
    if ((threadIdx.x & 31) == 0) {
        if (lp != 0.0) atomicAdd(logp, lp);
        if (ncand) atomicAdd(&ctrl->pair_tests, (unsigned long long)ncand);  // potential edges of this sample
        if (nedge) atomicAdd(&ctrl->edges, (unsigned long long)nedge);       // sampled edges
    }
}

static inline unsigned int blocks_for(int64_t n, int per_block) { return (unsigned int)((n + per_block - 1) / per_block); }

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
    if (grad && (e = cudaMemsetAsync(grad, 0, (size_t)N * 3 * sizeof(float), s)) != cudaSuccess) return e;
    StochParams sp;
    sp.b2 = b_link * b_link;
    sp.alpha = alpha;
    sp.gscale = -2.0 * (double)alpha / (double)sp.b2;
    sp.seed = seed;
    sp.sample = sample;
    iota_kernel<<<blocks_for(N, kBlock), kBlock, 0, s>>>(labels, N);
    link_stochastic_kernel<<<blocks_for(N, kBlock), kBlock, 0, s>>>(sorted, N, g, cell_start, idx_s, rel, sp, logp, grad,
                                                                    ctrl);
    return launch_write_labels(rel, idx_s, labels, N, s);
}

}  // namespace fof
