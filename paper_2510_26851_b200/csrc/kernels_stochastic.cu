// kernels_stochastic.cu — stochastic-edge Friends-of-Friends.
// PAPER.md section 3.2 (Eq. 6-8): every potential edge is y_ij ~ Bernoulli(p_ij),
// p_ij = sigma(alpha (b^2 - d_ij^2) / b^2); the halos of one Monte Carlo sample are the connected
// components of the sampled edges, and REINFORCE (Eq. 7) needs log p(y) and its gradient.
// Readings R25-R28 of DESIGN.md: potential edges = pairs within the candidate radius the plan was
// created with; sigma = the logistic evaluated by a fixed float32 recipe; counter-based randomness
// keyed on (seed, sample, original indices); d log p / d x_i = sum_j (y - p)(-2 alpha delta / b^2).
// The binning is NOT redone: the kernel walks the cell-sorted arrays that the last fof_link left in
// the workspace ("we do not rebuild the neighbor list", and S samples share one sort).
// One warp per 32 home particles; per stencil cell the candidate ranges are flattened across the warp.
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

// One warp per 32 consecutive cell-sorted home particles, one per lane.  For each of the 27 stencil
// cells in turn, the lanes' candidate ranges (reach-filtered) are flattened into slots that the 32
// lanes walk together, so a home particle in a dense cell does not serialise its warp.  A pair is
// "owned" (counted, added to log p, hooked) by the particle that sees the other one later in its
// own cell or in its forward half stencil; seen from the other side the same pair (same p, same y:
// the generator is keyed on the pair) only feeds the home particle's gradient.  The gradient terms
// of one batch are summed per home particle by a segmented warp scan (slots of one home particle
// are consecutive) and kept in shared memory: no atomics, fixed summation order.
constexpr int kStochWarps = kBlock / 32;

__global__ void __launch_bounds__(kBlock) link_stochastic_kernel(const float4 *__restrict__ sorted, int64_t N, Grid g,
                                                                 const unsigned int *__restrict__ cs,
                                                                 const int *__restrict__ idx_s, unsigned int *rel,
                                                                 StochParams sp, double *logp, float *grad,
                                                                 Ctrl *ctrl)
{
    __shared__ float s_g[kStochWarps][32][3];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int64_t s64 = ((int64_t)blockIdx.x * kStochWarps + wib) * 32 + lane;
    const bool valid = s64 < N;
    const int si = (int)min(s64, N - 1);
    const float4 me = __ldg(sorted + si);
    const unsigned int oi = (unsigned int)__ldg(idx_s + si);
    const int n = g.n;
    const float ux = __fmul_rn(me.x, g.inv_cell), uy = __fmul_rn(me.y, g.inv_cell), uz = __fmul_rn(me.z, g.inv_cell);
    const int cx = min(__float2int_rd(ux), g.n_minus_1), cy = min(__float2int_rd(uy), g.n_minus_1),
              cz = min(__float2int_rd(uz), g.n_minus_1);
    const float fx = ux - (float)cx, fy = uy - (float)cy, fz = uz - (float)cz;
    const float lo = g.reach, hi = 1.0f - g.reach;
    float lp = 0.0f;  // a lane adds at most a few thousand O(1) terms: float32 is enough before the float64 reduction
    unsigned int ncand = 0, nedge = 0;
    s_g[wib][lane][0] = s_g[wib][lane][1] = s_g[wib][lane][2] = 0.0f;
    __syncwarp();
    int dx = -2, dy = -1, dz = -1;
    for (int q = 0; q < 27; ++q) {
        if (++dx > 1) { dx = -1; if (++dy > 1) { dy = -1; ++dz; } }  // q = (dx + 1) + 3 (dy + 1) + 9 (dz + 1)
        const bool forward = q > 13;  // dz > 0, or dz == 0 and dy > 0, or dz == dy == 0 and dx > 0
        if (!forward && q != 13 && !grad) continue;  // the backward half only feeds the gradient
        int beg = 0, len = 0;
        if (valid && !((dx < 0 && !(fx < lo)) || (dx > 0 && !(fx > hi)) || (dy < 0 && !(fy < lo)) ||
                       (dy > 0 && !(fy > hi)) || (dz < 0 && !(fz < lo)) || (dz > 0 && !(fz > hi)))) {
            int ax = cx + dx, ay = cy + dy, az = cz + dz;
            ax = ax < 0 ? n - 1 : (ax >= n ? 0 : ax);
            ay = ay < 0 ? n - 1 : (ay >= n ? 0 : ay);
            az = az < 0 ? n - 1 : (az >= n ? 0 : az);
            const unsigned int c = cell_id(ax, ay, az, n);
            beg = (int)__ldg(cs + c);
            len = (int)__ldg(cs + c + 1) - beg;
        }
        int incl = len;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += v;
        }
        const int total = __shfl_sync(0xffffffffu, incl, 31);
        const int excl = incl - len;
        for (int p0 = 0; p0 < total; p0 += 32) {
            const int p = p0 + lane;
            const bool has = p < total;
            int owner = 0;  // the first lane whose inclusive prefix exceeds p
#pragma unroll
            for (int st = 16; st > 0; st >>= 1) {
                const int v = __shfl_sync(0xffffffffu, incl, owner + st - 1);
                if (v <= p) owner += st;
            }
            owner = min(owner, 31);
            const int j = __shfl_sync(0xffffffffu, beg, owner) + (p - __shfl_sync(0xffffffffu, excl, owner));
            const float ox = __shfl_sync(0xffffffffu, me.x, owner), oy = __shfl_sync(0xffffffffu, me.y, owner),
                        oz = __shfl_sync(0xffffffffu, me.z, owner);
            const int osi = __shfl_sync(0xffffffffu, si, owner);
            const unsigned int ooi = __shfl_sync(0xffffffffu, oi, owner);
            float gx = 0.0f, gy = 0.0f, gz = 0.0f;
            if (has && j != osi) {
                const float4 pj = __ldg(sorted + j);
                const float ddx = min_image(__fsub_rn(ox, pj.x), g.L, g.h);
                const float ddy = min_image(__fsub_rn(oy, pj.y), g.L, g.h);
                const float ddz = min_image(__fsub_rn(oz, pj.z), g.L, g.h);
                const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(ddx, ddx), __fmul_rn(ddy, ddy)), __fmul_rn(ddz, ddz));
                if (d2 <= g.b2) {  // R25: beyond the candidate radius p = 0
                    const float tt = __fmul_rn(sp.c, __fsub_rn(sp.b2, d2));
                    float e;
                    const float pr = sigmoid_fixed(tt, e);
                    const unsigned int oj = (unsigned int)__ldg(idx_s + j);
                    const float u = __fmul_rn((float)rng_u24(sp.key, min(ooi, oj), max(ooi, oj)), 5.9604644775390625e-8f);
                    const bool y = u < pr;
                    const float tc = fminf(fmaxf(tt, -30.0f), 30.0f);
                    if (grad && tt == tc) {
                        const float cgr = ((y ? 1.0f : 0.0f) - pr) * sp.gscale;
                        gx = cgr * ddx;
                        gy = cgr * ddy;
                        gz = cgr * ddz;
                    }
                    if (forward || (q == 13 && j > osi)) {
                        ++ncand;
                        // log p = -log(1 + e); log(1 - p) = log(e / (1 + e)) = log p - t; float32 terms
                        lp += -__logf(__fadd_rn(1.0f, e)) - (y ? 0.0f : tc);
                        if (y) {
                            ++nedge;
                            const int pa = osi - (int)rel[osi], pb = j - (int)rel[j];
                            if (pa != pb) unite_rel(rel, idx_s, osi, j);  // same parent: already one set
                        }
                    }
                }
            }
            if (grad && __any_sync(0xffffffffu, gx != 0.0f || gy != 0.0f || gz != 0.0f)) {
                // segmented inclusive scan over runs of equal owner, then one add per home particle
                const int key = has ? owner : -1 - lane;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const float vx = __shfl_up_sync(0xffffffffu, gx, o), vy = __shfl_up_sync(0xffffffffu, gy, o),
                                vz = __shfl_up_sync(0xffffffffu, gz, o);
                    const int k = __shfl_up_sync(0xffffffffu, key, o);
                    if (lane >= o && k == key) { gx += vx; gy += vy; gz += vz; }
                }
                const int knext = __shfl_down_sync(0xffffffffu, key, 1);
                if (has && (lane == 31 || knext != key)) {
                    s_g[wib][owner][0] += gx;
                    s_g[wib][owner][1] += gy;
                    s_g[wib][owner][2] += gz;
                }
                __syncwarp();
            }
        }
    }
    __syncwarp();
    if (grad && valid) {
        grad[3 * (int64_t)oi + 0] = s_g[wib][lane][0];
        grad[3 * (int64_t)oi + 1] = s_g[wib][lane][1];
        grad[3 * (int64_t)oi + 2] = s_g[wib][lane][2];
    }
    double lpd = (double)lp;
    for (int o = 16; o > 0; o >>= 1) {
        lpd += __shfl_xor_sync(0xffffffffu, lpd, o);
        ncand += __shfl_xor_sync(0xffffffffu, ncand, o);
        nedge += __shfl_xor_sync(0xffffffffu, nedge, o);
    }
    if (lane == 0) {
        if (lpd != 0.0) atomicAdd(logp, lpd);
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
    StochParams sp;
    sp.b2 = b_link * b_link;
    sp.c = alpha / sp.b2;
    sp.gscale = -2.0f * sp.c;
    unsigned int k = (unsigned int)(seed ^ (seed >> 32)) ^ (sample * 0x9E3779B9U);  // per-sample key: mix32 on the host
    k ^= k >> 16; k *= 0x7FEB352DU;
    k ^= k >> 15; k *= 0x846CA68BU;
    k ^= k >> 16;
    sp.key = k;
    iota_kernel<<<blocks_for(N, kBlock), kBlock, 0, s>>>(labels, N);
    link_stochastic_kernel<<<blocks_for(N, kBlock), kBlock, 0, s>>>(sorted, N, g, cell_start, idx_s, rel, sp, logp, grad,
                                                                    ctrl);
    return launch_write_labels(rel, idx_s, labels, N, s);
}

}  // namespace fof
