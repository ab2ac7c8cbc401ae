// kernels_link.cu — H4 half-stencil pair tests + union, H5 flatten.
// What is linked: PAPER.md:85-87 (§2 step iv) and PAPER.md:200-214 (Alg. 2 candidate cells and
// mask); the 27-cell stencil with indices mod n is PAPER.md:202.  The T label sweeps of
// PAPER.md:221-225 are replaced by their fixed point, computed with a lock-free union-find on the
// label array (root = minimum original index = the converged min-label).
#include "fof_internal.cuh"

namespace fof {

// Half stencil: every unordered pair of distinct neighbouring cells is visited from exactly one
// side (needs n >= 3 so that +1 and -1 are different cells).  Rows (dy, dz) of three x-adjacent
// cells, then the +x neighbour in the home row, then the home cell itself (j > i).
__constant__ int kRowDy[4] = {-1, 0, 1, 1};
__constant__ int kRowDz[4] = {1, 1, 1, 0};

struct PairCounters {
    unsigned int edges;
    unsigned int tests;
};

__device__ __forceinline__ void test_range(const float4 *__restrict__ sorted, unsigned int beg, unsigned int end,
                                           const float4 me, int oi, const Grid &g, int *parent, PairCounters &pc)
{
    pc.tests += end - beg;
    for (unsigned int t = beg; t < end; ++t) {
        const float4 pj = __ldg(sorted + t);
        if (linked(me.x, me.y, me.z, pj.x, pj.y, pj.z, g)) {
            ++pc.edges;
            const int oj = __float_as_int(pj.w);
            // already in one set?  (a stale parent is still a member of the same set: safe to skip)
            if (parent[oi] != parent[oj]) unite(parent, oi, oj);
        }
    }
}

// V1: one thread per cell-sorted particle.
__global__ void __launch_bounds__(kBlock) link_kernel(const float4 *__restrict__ sorted, int64_t N, Grid g,
                                                      const unsigned int *__restrict__ cell_start, int *parent,
                                                      Ctrl *ctrl)
{
    const int64_t s = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    PairCounters pc = {0u, 0u};
    if (s < N) {
        const float4 me = __ldg(sorted + s);
        const int oi = __float_as_int(me.w);
        const int n = g.n;
        const int cx = cell1(me.x, g), cy = cell1(me.y, g), cz = cell1(me.z, g);
        const int xm = cx == 0 ? n - 1 : cx - 1, xp = cx == n - 1 ? 0 : cx + 1;
        const bool interior = (cx > 0) && (cx < n - 1);
        // home cell: partners after me; then the +x cell
        const unsigned int home = cell_id(cx, cy, cz, n);
        if (interior) {
            test_range(sorted, (unsigned int)s + 1, __ldg(cell_start + home + 2), me, oi, g, parent, pc);
        } else {
            test_range(sorted, (unsigned int)s + 1, __ldg(cell_start + home + 1), me, oi, g, parent, pc);
            const unsigned int c = cell_id(xp, cy, cz, n);
            test_range(sorted, __ldg(cell_start + c), __ldg(cell_start + c + 1), me, oi, g, parent, pc);
        }
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            int ny = cy + kRowDy[r], nz = cz + kRowDz[r];
            ny = ny < 0 ? n - 1 : (ny >= n ? 0 : ny);
            nz = nz >= n ? 0 : nz;
            if (interior) {
                const unsigned int c = cell_id(cx - 1, ny, nz, n);
                test_range(sorted, __ldg(cell_start + c), __ldg(cell_start + c + 3), me, oi, g, parent, pc);
            } else {
                const int xs[3] = {xm, cx, xp};
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    const unsigned int c = cell_id(xs[k], ny, nz, n);
                    test_range(sorted, __ldg(cell_start + c), __ldg(cell_start + c + 1), me, oi, g, parent, pc);
                }
            }
        }
    }
    // per-warp totals -> two atomics per warp
    unsigned long long e = pc.edges, t = pc.tests;
    for (int o = 16; o > 0; o >>= 1) {
        e += __shfl_xor_sync(0xffffffffu, e, o);
        t += __shfl_xor_sync(0xffffffffu, t, o);
    }
    if ((threadIdx.x & 31) == 0 && t) {
        if (e) atomicAdd(&ctrl->edges, e);
        atomicAdd(&ctrl->pair_tests, t);
    }
}

// H5: labels[i] <- root(i), in place ("after convergence").  A concurrent reader
// sees either the old parent (an ancestor) or the root: both lead to the same root.
__global__ void __launch_bounds__(kBlock) flatten_kernel(int *labels, int64_t N)
{
    const int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (i >= N) return;
    int r = labels[i];
    if (r == (int)i) return;
    int p = labels[r];
    while (p != r) { r = p; p = labels[r]; }
    labels[i] = r;
}

static inline unsigned int blocks_for(int64_t n, int per_block) { return (unsigned int)((n + per_block - 1) / per_block); }

cudaError_t launch_link(const float4 *sorted, int64_t N, Grid g, const unsigned int *cell_start, int *labels,
                        Ctrl *ctrl, int num_sms, cudaStream_t s)
{
    (void)num_sms;
    if (N > 0) link_kernel<<<blocks_for(N, kBlock), kBlock, 0, s>>>(sorted, N, g, cell_start, labels, ctrl);
    return cudaGetLastError();
}

cudaError_t launch_flatten(int *labels, int64_t N, cudaStream_t s)
{
    if (N > 0) flatten_kernel<<<blocks_for(N, kBlock), kBlock, 0, s>>>(labels, N);
    return cudaGetLastError();
}

}  // namespace fof
