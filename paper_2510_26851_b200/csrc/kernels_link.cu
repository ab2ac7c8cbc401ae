// kernels_link.cu — H4 half-stencil pair tests + union, H5 flatten + canonical labels.
// What is linked: PAPER.md:85-87 (§2 step iv) and PAPER.md:200-214 (Alg. 2 candidate cells and
// mask); the 27-cell stencil with indices mod n is PAPER.md:202.  The T label sweeps of
// PAPER.md:221-225 are replaced by their fixed point, computed with a lock-free union-find
// (ECL-CC style: atomicCAS hooks at roots, path halving) whose root is the minimum index of its
// set, the converged min-label of PAPER.md:91.
//
// Design.  The union-find runs in CELL-SORTED index space: a component is a
// spatially compact object, so its parent entries sit in a few cache lines and the "already in
// one set?" check of an edge is a coalesced / L1-resident load instead of a random access into
// a 4N-byte array.  One thread owns one cell-sorted particle and walks its (at most five)
// candidate ranges: the rest of its own cell (+ the +x cell), and the rows (dy,dz) = (+1,0),
// (-1,+1), (0,+1), (+1,+1), each a contiguous run of up to three cells of the sorted array.
// A geometric reach filter drops every neighbour cell that is farther than b from the particle.
// The canonical label (minimum ORIGINAL index of the component) is produced by two streaming
// passes: flatten + atomicMin of the original index at the root, then a scatter of that minimum
// to labels[original index].
#include "fof_internal.cuh"

namespace fof {

// ---- link predicate, with the minimum-image selects compiled out where they are provably
// no-ops (all tested pairs sit in adjacent, non-wrapping cells and n >= 6, so |d| < L/2): the bits
// of d2 are the same either way.
template <bool WRAP>
__device__ __forceinline__ bool linked_t(const float4 &a, const float4 &b, const Grid &g)
{
    float dx = __fsub_rn(a.x, b.x), dy = __fsub_rn(a.y, b.y), dz = __fsub_rn(a.z, b.z);
    if (WRAP) {
        dx = min_image(dx, g.L, g.h);
        dy = min_image(dy, g.L, g.h);
        dz = min_image(dz, g.L, g.h);
    }
    const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
    return d2 <= g.b2;
}

// ---- union-find on `rel`: rel[s] = s - parent(s) >= 0 (a root has rel 0, so the forest is
// initialised by a memset; the root of a set is its smallest cell-sorted index).  Hooks are
// atomicCAS(rel + root, 0, distance) and can only succeed on a true root; every plain load may
// return a stale value, which is always the offset to SOME ancestor (links only ever move up), so
// staleness costs hops, never correctness.  Plain path-halving stores at non-roots are benign.
__device__ __forceinline__ int find_rel(unsigned int *rel, int x)
{
    unsigned int d = rel[x];
    while (d) {
        const int p = x - (int)d;
        const unsigned int dp = rel[p];
        if (dp) rel[x] = d + dp;  // halve: x -> grandparent
        x = p;
        d = dp;
    }
    return x;
}

__device__ __forceinline__ int unite_rel(unsigned int *rel, int a, int b)
{
    int ra = find_rel(rel, a), rb = find_rel(rel, b);
    while (ra != rb) {
        if (ra < rb) { const int t = ra; ra = rb; rb = t; }  // ra is the larger root
        const unsigned int old = atomicCAS(rel + ra, 0u, (unsigned int)(ra - rb));
        if (old == 0u) return rb;
        ra = find_rel(rel, ra - (int)old);
    }
    return ra;
}

// One candidate range of one home particle.  `root` caches the home particle's current root.
template <bool WRAP>
__device__ __forceinline__ void test_range(const float4 *__restrict__ sorted, unsigned int *rel, int beg, int end,
                                           const float4 &me, int si, int &root, const Grid &g, unsigned int &edges)
{
    // four candidates per trip: all loads (positions and parent offsets) are issued before the first
    // test, so one memory latency covers four tests.  A parent offset read early may be stale after
    // a union in the same trip; that only costs a redundant find.
    for (int t = beg; t < end; t += 4) {
        float4 pj[4];
        unsigned int rj[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int tt = min(t + u, end - 1);
            pj[u] = __ldg(sorted + tt);
            rj[u] = rel[tt];
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int tt = t + u;
            if (tt < end && linked_t<WRAP>(me, pj[u], g)) {
                ++edges;
                if (tt - (int)rj[u] != root) {  // not yet known to be in one set
                    root = unite_rel(rel, si, tt);
                    if (si != root) rel[si] = (unsigned int)(si - root);
                    if (tt != root) rel[tt] = (unsigned int)(tt - root);
                }
            }
        }
    }
}

// Everything thread `si` needs to know about its candidates.
struct Home {
    int cx, cy, cz;
    bool xl, xh, yl, yh, zh;  // within `reach` of the low / high face of its cell
};

// Row (y', z') of the grid, cells [cx - xl, cx + 1 + xh) clipped to the row: one run of `sorted`.
// The cells reached through the periodic x faces are handled by wrapped_pieces().
template <bool WRAP>
__device__ __forceinline__ void row_range(const unsigned int *__restrict__ cs, const Home &h, int yy, int zz, int n,
                                          bool with_lower, int &beg, int &end)
{
    const int rb = n * (yy + n * zz);
    const int a = max(h.cx - (with_lower && h.xl ? 1 : 0), 0);
    const int b = min(h.cx + 1 + (h.xh ? 1 : 0), n);
    beg = (int)__ldg(cs + rb + a);
    end = (int)__ldg(cs + rb + b);
}

// ---- warp-level work distribution.  The candidate ranges of the 32 home particles of a warp are
// cut into chunks of at most kChunk candidates, queued in shared memory, and handed out to the
// lanes round-robin, so that a lane sitting in a dense cell does not hold 31 idle lanes hostage.
constexpr int kChunk = 8;                 // candidates per chunk
constexpr int kQueue = 256;               // chunks per warp and window
constexpr int kWarpsPerCta = kLinkBlock / 32;

template <bool WRAP>
__device__ __forceinline__ void warp_link(const float4 *__restrict__ sorted, const unsigned int *__restrict__ cs,
                                          unsigned int *rel, int si, bool valid, const float4 &me, const Home &h,
                                          const Grid &g, int2 *q, unsigned int &edges, unsigned int &tests)
{
    constexpr int NR = WRAP ? 10 : 5;
    const int n = g.n;
    const int lane = threadIdx.x & 31;
    int beg[NR], len[NR];
#pragma unroll
    for (int k = 0; k < NR; ++k) beg[k] = len[k] = 0;
    if (valid) {
        int yp = h.cy + 1, ym = h.cy - 1, zp = h.cz + 1;
        if (WRAP) {
            if (yp == n) yp = 0;
            if (ym < 0) ym = n - 1;
            if (zp == n) zp = 0;
        }
        int e;
        // home row: the rest of my cell, plus the +x cell
        // (the pairs inside a DENSE home cell belong to link_dense_kernel)
        {
            const unsigned int *row = cs + n * (h.cy + n * h.cz) + h.cx;
            const int c0 = (int)__ldg(row), c1 = (int)__ldg(row + 1);
            const int e0 = (h.xh && h.cx + 1 < n) ? (int)__ldg(row + 2) : c1;
            beg[0] = (c1 - c0 >= kDenseCell && c1 - c0 <= kDenseMax) ? c1 : si + 1;
            len[0] = e0 - beg[0];
        }
        if (h.yh) { row_range<WRAP>(cs, h, yp, h.cz, n, true, beg[1], e); len[1] = e - beg[1]; }
        if (h.zh) {
            row_range<WRAP>(cs, h, h.cy, zp, n, true, beg[2], e); len[2] = e - beg[2];
            if (h.yl) { row_range<WRAP>(cs, h, ym, zp, n, true, beg[3], e); len[3] = e - beg[3]; }
            if (h.yh) { row_range<WRAP>(cs, h, yp, zp, n, true, beg[4], e); len[4] = e - beg[4]; }
        }
        if (WRAP) {
            // cells behind the periodic x faces: cell 0 of a row when cx = n-1 reaches up, cell n-1
            // when cx = 0 reaches down (never for the home row's lower side: half stencil)
            const bool up = h.xh && h.cx == n - 1, dn = h.xl && h.cx == 0;
            if (up || dn) {
                const int ys[5] = {h.cy, yp, h.cy, ym, yp};
                const int zs[5] = {h.cz, h.cz, zp, zp, zp};
                const bool on[5] = {true, h.yh, h.zh, h.zh && h.yl, h.zh && h.yh};
#pragma unroll
                for (int k = 0; k < 5; ++k) {
                    if (!on[k] || (!up && k == 0)) continue;
                    // up and dn exclude each other unless n == 1 row cell... (n >= 3: cx cannot be both)
                    const int c = n * (ys[k] + n * zs[k]) + (up ? 0 : n - 1);
                    beg[5 + k] = (int)__ldg(cs + c);
                    len[5 + k] = (int)__ldg(cs + c + 1) - beg[5 + k];
                }
            }
        }
    }
    int nch = 0;
#pragma unroll
    for (int k = 0; k < NR; ++k) nch += (len[k] + kChunk - 1) / kChunk;
    int incl = nch;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
    }
    const int total = __shfl_sync(0xffffffffu, incl, 31);
    const int excl = incl - nch;
    for (int base = 0; base < total; base += kQueue) {
        int pos = excl - base;
#pragma unroll
        for (int k = 0; k < NR; ++k)
            for (int o = 0; o < len[k]; o += kChunk, ++pos)
                if (pos >= 0 && pos < kQueue) q[pos] = make_int2(beg[k] + o, (min(kChunk, len[k] - o) << 8) | lane);
        __syncwarp();
        const int cnt = min(kQueue, total - base);
        for (int j0 = 0; j0 < cnt; j0 += 32) {
            const int j = j0 + lane;
            const bool has = j < cnt;
            const int2 c = has ? q[j] : make_int2(0, lane);
            const int owner = c.y & 31;
            float4 o4;
            o4.x = __shfl_sync(0xffffffffu, me.x, owner);
            o4.y = __shfl_sync(0xffffffffu, me.y, owner);
            o4.z = __shfl_sync(0xffffffffu, me.z, owner);
            o4.w = 0.0f;
            const int osi = __shfl_sync(0xffffffffu, si, owner);
            if (has) {
                const int cb = c.x, ce = c.x + (c.y >> 8);
                tests += (unsigned int)(ce - cb);
                int root = osi - (int)rel[osi];
                test_range<WRAP>(sorted, rel, cb, ce, o4, osi, root, g, edges);
            }
        }
        __syncwarp();
    }
}

// H4.  Persistent grid: each CTA walks chunks of kLinkBlock consecutive cell-sorted particles.
__global__ void __launch_bounds__(kLinkBlock) link_kernel(const float4 *__restrict__ sorted, int64_t N, Grid g,
                                                          const unsigned int *__restrict__ cell_start,
                                                          unsigned int *rel, Ctrl *ctrl)
{
    __shared__ int2 s_queue[kWarpsPerCta][kQueue];
    int2 *q = s_queue[threadIdx.x >> 5];
    unsigned int edges = 0, tests = 0;
    const int n = g.n;
    const float lo = g.reach, hi = 1.0f - g.reach;
    for (int64_t base = (int64_t)blockIdx.x * kLinkBlock; base < N; base += (int64_t)gridDim.x * kLinkBlock) {
        const int64_t s64 = base + threadIdx.x;
        const bool valid = s64 < N;
        const int si = (int)s64;
        float4 me = make_float4(0.f, 0.f, 0.f, 0.f);
        Home h;
        bool needwrap = false;
        if (valid) {
            me = __ldg(sorted + si);
            const float ux = __fmul_rn(me.x, g.inv_cell), uy = __fmul_rn(me.y, g.inv_cell),
                        uz = __fmul_rn(me.z, g.inv_cell);
            h.cx = min(__float2int_rd(ux), g.n_minus_1);
            h.cy = min(__float2int_rd(uy), g.n_minus_1);
            h.cz = min(__float2int_rd(uz), g.n_minus_1);
            const float fx = ux - (float)h.cx, fy = uy - (float)h.cy, fz = uz - (float)h.cz;
            h.xl = fx < lo; h.xh = fx > hi;
            h.yl = fy < lo; h.yh = fy > hi;
            h.zh = fz > hi;
            needwrap = n < 6 || (h.xl && h.cx == 0) || (h.xh && h.cx == n - 1) || (h.yl && h.cy == 0) ||
                       (h.yh && h.cy == n - 1) || (h.zh && h.cz == n - 1);
        }
        if (__any_sync(0xffffffffu, needwrap)) warp_link<true>(sorted, cell_start, rel, si, valid, me, h, g, q, edges, tests);
        else warp_link<false>(sorted, cell_start, rel, si, valid, me, h, g, q, edges, tests);
    }
    for (int o = 16; o > 0; o >>= 1) {
        edges += __shfl_xor_sync(0xffffffffu, edges, o);
        tests += __shfl_xor_sync(0xffffffffu, tests, o);
    }
    if ((threadIdx.x & 31) == 0) {  // one pair of global atomics per warp: no CTA barrier at the end
        if (edges) atomicAdd(&ctrl->edges, (unsigned long long)edges);
        if (tests) atomicAdd(&ctrl->pair_tests, (unsigned long long)tests);
    }
}

// H4 (dense cells): all pairs inside one cell that holds kDenseCell..kDenseMax particles, one warp
// per cell, run BEFORE link_kernel (every parent entry of the cell is still a root and no other
// warp touches it).  The cell is cut into blocks of 32 particles.  For a tile (block I, block J <= I)
// lane i builds the adjacency bitmask of its particle against the 32 particles of J with
// warp-uniform loads (one transaction per candidate, 32 tests per trip).  Diagonal tile: the
// components of the 32-node graph are closed by squaring the reachability masks through shuffles,
// and written as parent offsets with plain stores -- no atomics.  Off-diagonal tile: the masks are
// reduced to (component of I, component of J) pairs and only those are united.
// Pairs inside one cell never wrap (cell side <= L/3 < L/2).
__global__ void __launch_bounds__(kLinkBlock) link_dense_kernel(const float4 *__restrict__ sorted, Grid g,
                                                                const unsigned int *__restrict__ cell_start,
                                                                const unsigned int *__restrict__ dense_list,
                                                                unsigned int *rel, Ctrl *ctrl)
{
    __shared__ unsigned char s_lab_all[kWarpsPerCta][kDenseMax];
    __shared__ float4 s_pj_all[kWarpsPerCta][32];
    unsigned char *s_lab = s_lab_all[threadIdx.x >> 5];
    float4 *s_pj = s_pj_all[threadIdx.x >> 5];
    const int lane = threadIdx.x & 31;
    const unsigned int nd = ctrl->ndense;
    const unsigned int nwarps = gridDim.x * kWarpsPerCta;
    const float inf = __int_as_float(0x7f800000);
    unsigned int edges = 0, tests = 0;
    for (unsigned int ci = blockIdx.x * kWarpsPerCta + (threadIdx.x >> 5); ci < nd; ci += nwarps) {
        const unsigned int c = __ldg(dense_list + ci);
        const int b0 = (int)__ldg(cell_start + c), e0 = (int)__ldg(cell_start + c + 1);
        for (int ib = b0; ib < e0; ib += 32) {
            const int i = ib + lane;
            const bool valid = i < e0;
            // a lane without a particle sits at +inf: d2 = inf fails the test on both sides of a tile
            float4 me = make_float4(inf, inf, inf, 0.0f);
            if (valid) me = __ldg(sorted + i);
            int lab = lane;  // lane of the smallest member of my component inside block I
            for (int jb = ib; jb >= b0; jb -= 32) {  // diagonal tile first, then the earlier blocks
                // block J staged in shared memory: the tile loop reads it with broadcast LDS.128
                __syncwarp();
                s_pj[lane] = (jb == ib) ? me : __ldg(sorted + jb + lane);  // earlier blocks are full
                __syncwarp();
                const int cnt = min(32, e0 - jb);
                unsigned int adj = 0;
#pragma unroll 1
                for (int j0 = 0; j0 < cnt; j0 += 8) {
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        if (linked_t<false>(me, s_pj[j0 + u], g)) adj |= 1u << (j0 + u);
                }
                if (jb == ib) {
                    adj &= ~(1u << lane);
                    edges += (unsigned int)__popc(adj & ((1u << lane) - 1u));
                    if (valid) tests += (unsigned int)lane;
                    // components of the 32-node graph: breadth-first from the lowest unlabelled lane; one
                    // REDUX (warp OR of the visited lanes' adjacency) per BFS level
                    const unsigned int self = 1u << lane;
                    unsigned int todo = 0xffffffffu;
                    while (todo) {
                        const int r = __ffs((int)todo) - 1;
                        unsigned int vis = 1u << r;
                        while (true) {
                            const unsigned int nxt = vis | __reduce_or_sync(0xffffffffu, (vis & self) ? adj : 0u);
                            if (nxt == vis) break;
                            vis = nxt;
                        }
                        if (vis & self) lab = r;
                        todo &= ~vis;
                    }
                    if (valid && lab != lane) rel[i] = (unsigned int)(lane - lab);
                    s_lab[i - b0] = (unsigned char)lab;
                } else {
                    edges += (unsigned int)__popc(adj);
                    if (valid) tests += 32u;
                    unsigned int reps = 0;
                    for (unsigned int m = adj; m; m &= m - 1u) reps |= 1u << s_lab[jb - b0 + __ffs((int)m) - 1];
                    const unsigned int peers = __match_any_sync(0xffffffffu, lab);
                    reps = __reduce_or_sync(peers, reps);
                    if (lane == lab)
                        for (unsigned int m = reps; m; m &= m - 1u) unite_rel(rel, i, jb + __ffs((int)m) - 1);
                }
            }
        }
        __syncwarp();
    }
    for (int o = 16; o > 0; o >>= 1) {
        edges += __shfl_xor_sync(0xffffffffu, edges, o);
        tests += __shfl_xor_sync(0xffffffffu, tests, o);
    }
    if (lane == 0) {
        if (edges) atomicAdd(&ctrl->edges, (unsigned long long)edges);
        if (tests) atomicAdd(&ctrl->pair_tests, (unsigned long long)tests);
    }
}

// H5a: flatten ("after convergence"): rel[s] <- s - root(s), and lower the root's
// minidx to the smallest ORIGINAL index of its members ("minimum label", PAPER.md:180
// "minimum global particle ID").  The chase is read-only; a concurrent reader sees either the old
// offset (an ancestor) or the root.  Roots have nothing to do: minidx[root] starts as its own index.
__global__ void __launch_bounds__(kBlock) flatten_min_kernel(unsigned int *rel, const int *__restrict__ idx_s,
                                                             int *minidx, int64_t N)
{
    const int64_t s = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (s >= N) return;
    unsigned int d = rel[s];
    if (d == 0u) return;
    int r = (int)s - (int)d;
    while ((d = rel[r]) != 0u) r -= (int)d;
    rel[s] = (unsigned int)((int)s - r);
    atomicMin(minidx + r, idx_s[s]);
}

// H5b: labels[original index] = minimum original index of the component.
__global__ void __launch_bounds__(kBlock) write_labels_kernel(const unsigned int *__restrict__ rel,
                                                              const int *__restrict__ idx_s,
                                                              const int *__restrict__ minidx, int *__restrict__ labels,
                                                              int64_t N)
{
    const int64_t s = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (s >= N) return;
    const int r = (int)s - (int)__ldg(rel + s);
    labels[__ldg(idx_s + s)] = __ldg(minidx + r);
}

// P_exec of DESIGN.md §7: candidate pairs the unfiltered half stencil implies on this grid,
// sum over cells of occ (occ - 1) / 2 + occ * (occupancy of the 13 half-stencil cells).  Run by
// fof_link_stats only (not on the hot path).
__constant__ int kRowDy[4] = {-1, 0, 1, 1};
__constant__ int kRowDz[4] = {1, 1, 1, 0};

__global__ void __launch_bounds__(kBlock) grid_pairs_kernel(const unsigned int *__restrict__ cell_start, Grid g,
                                                            Ctrl *ctrl)
{
    const int n = g.n;
    const int64_t C = (int64_t)n * n * n;
    unsigned long long sum = 0;
    for (int64_t c = (int64_t)blockIdx.x * kBlock + threadIdx.x; c < C; c += (int64_t)gridDim.x * kBlock) {
        const unsigned long long occ = cell_start[c + 1] - cell_start[c];
        if (!occ) continue;
        const int cx = (int)(c % n), cy = (int)((c / n) % n), cz = (int)(c / ((int64_t)n * n));
        const int xm = cx == 0 ? n - 1 : cx - 1, xp = cx == n - 1 ? 0 : cx + 1;
        unsigned long long nb = 0;
        { const unsigned int d = cell_id(xp, cy, cz, n); nb += cell_start[d + 1] - cell_start[d]; }
        for (int r = 0; r < 4; ++r) {
            int ny = cy + kRowDy[r], nz = cz + kRowDz[r];
            ny = ny < 0 ? n - 1 : (ny >= n ? 0 : ny);
            nz = nz >= n ? 0 : nz;
            const int xs[3] = {xm, cx, xp};
            for (int k = 0; k < 3; ++k) { const unsigned int d = cell_id(xs[k], ny, nz, n); nb += cell_start[d + 1] - cell_start[d]; }
        }
        sum += occ * (occ - 1) / 2 + occ * nb;
    }
    for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
    if ((threadIdx.x & 31) == 0 && sum) atomicAdd(&ctrl->grid_pairs, sum);
}

cudaError_t launch_grid_pairs(const unsigned int *cell_start, Grid g, Ctrl *ctrl, int num_sms, cudaStream_t s)
{
    grid_pairs_kernel<<<(unsigned int)(num_sms > 0 ? num_sms * 8 : 1024), kBlock, 0, s>>>(cell_start, g, ctrl);
    return cudaGetLastError();
}

static inline unsigned int blocks_for(int64_t n, int per_block) { return (unsigned int)((n + per_block - 1) / per_block); }

cudaError_t launch_link(const float4 *sorted, int64_t N, Grid g, const unsigned int *cell_start,
                        const unsigned int *dense_list, unsigned int *rel, Ctrl *ctrl, int num_sms, cudaStream_t s)
{
    if (N <= 0) return cudaSuccess;
    const unsigned int grid = (unsigned int)min((int64_t)blocks_for(N, kLinkBlock), (int64_t)num_sms * 32);
    link_dense_kernel<<<(unsigned int)num_sms * 8, kLinkBlock, 0, s>>>(sorted, g, cell_start, dense_list, rel, ctrl);
    link_kernel<<<grid, kLinkBlock, 0, s>>>(sorted, N, g, cell_start, rel, ctrl);
    return cudaGetLastError();
}

cudaError_t launch_flatten_min(unsigned int *rel, const int *idx_s, int *minidx, int64_t N, cudaStream_t s)
{
    if (N > 0) flatten_min_kernel<<<blocks_for(N, kBlock), kBlock, 0, s>>>(rel, idx_s, minidx, N);
    return cudaGetLastError();
}

cudaError_t launch_write_labels(const unsigned int *rel, const int *idx_s, const int *minidx, int *labels, int64_t N,
                                cudaStream_t s)
{
    if (N > 0) write_labels_kernel<<<blocks_for(N, kBlock), kBlock, 0, s>>>(rel, idx_s, minidx, labels, N);
    return cudaGetLastError();
}

}  // namespace fof
