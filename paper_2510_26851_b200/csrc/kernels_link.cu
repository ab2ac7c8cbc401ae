// kernels_link.cu — H4 half-stencil pair tests + union, H5 flatten + canonical labels.
// What is linked: PAPER.md:85-87 (§2 step iv) and PAPER.md:200-214 (Alg. 2 candidate cells and
// mask); the 27-cell stencil with indices mod n is PAPER.md:202.  The T label sweeps of
// PAPER.md:221-225 are replaced by their fixed point, computed with a lock-free union-find
// (ECL-CC style: atomicCAS hooks at roots, path halving) whose root is the minimum index of its
// set, the converged min-label of PAPER.md:91.
//
// Design.  The union-find runs in CELL-SORTED index space: a component is a
// spatially compact object, so its parent entries sit in a few cache lines.  Every unordered
// pair of particles in the same or in adjacent cells is tested exactly once, by one of two kernels:
//   link_tiles_kernel   pairs with at least one particle in a DENSE cell (>= kDenseCell particles).
//                       One warp per (dense cell, tile of <= 32 of its particles): the tile sits in
//                       registers, one particle per lane; the candidates (the tile itself, the
//                       earlier tiles of the cell, and the particles of the 26 neighbour cells that
//                       lie within b of the cell) are staged 32 at a time in shared memory and
//                       broadcast, so one trip of 11 instructions tests 32 pairs.  The adjacency
//                       comes out as ballot bitmasks; components of the tile are closed in registers
//                       and only one hook per (component, adjacent candidate) reaches the union-find.
//                       A pair of two dense cells belongs to the one that sees the other in its
//                       forward half stencil.
//   link_sparse_kernel  pairs of two sparse cells.  One thread per particle collects its candidate
//                       ranges (own cell after itself + the 13 forward cells, reach-filtered);
//                       the ranges of a warp are flattened into one list of candidate slots that
//                       the 32 lanes walk together, so a lane with many candidates does not hold
//                       the others hostage.
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

// ---- union-find on `rel`: rel[s] = s - parent(s) >= 0 (a root has rel 0; the root of a set is
// its smallest cell-sorted index).  Hooks are atomicCAS(rel + root, 0, distance) and can only
// succeed on a true root; every plain load may return a stale value, which is always the offset
// to SOME ancestor (links only ever move up), so staleness costs hops, never correctness.  Plain
// path-halving stores at non-roots are benign.
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

constexpr int kWarpsPerCta = kLinkBlock / 32;
constexpr unsigned int kFull = 0xffffffffu;

__device__ __forceinline__ unsigned int lanemask_lt()
{
    unsigned int m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// =============================================================================================
// link_tiles_kernel: pairs that involve a dense cell.
// =============================================================================================

// Tile I (one particle per lane, `me`; idle lanes sit at +inf) against a batch of `cnt` <= 32
// candidates staged in shared memory.  Returns, in lane k, the mask of tile lanes linked to
// candidate k; `nedges` (warp-uniform) counts the set bits of all masks.
template <bool WRAP>
__device__ __forceinline__ unsigned int batch_adjacency(const float4 &me, const float4 *s_pj, int cnt, const Grid &g,
                                                        int lane, unsigned int &nedges)
{
    unsigned int adjT = 0;
#pragma unroll 4
    for (int k = 0; k < cnt; ++k) {
        const unsigned int bal = __ballot_sync(kFull, linked_t<WRAP>(me, s_pj[k], g));
        if (lane == k) adjT = bal;
        nedges += (unsigned int)__popc(bal);
    }
    return adjT;
}

// Hooks of one batch: candidate k (cell-sorted index in s_pj[k].w) joins every component of the
// tile it is linked to.  `grp` = lanes of my tile component, `leader` = I am its lowest lane.
__device__ __forceinline__ void batch_unions(unsigned int adjT, const float4 *s_pj, int cnt, unsigned int *rel, int ib,
                                             unsigned int grp, bool leader, int lane)
{
    const unsigned int active = __reduce_or_sync(kFull, adjT);  // tile lanes with any link into the batch
    if (!active) return;
    unsigned int lead = __ballot_sync(kFull, leader && (grp & active));
    const int j = (lane < cnt) ? __float_as_int(s_pj[lane].w) : 0;
    while (lead) {
        const int gl = __ffs((int)lead) - 1;
        lead &= lead - 1u;
        const unsigned int members = __shfl_sync(kFull, grp, gl);
        if (adjT & members) unite_rel(rel, j, ib + gl);
    }
}

// Neighbour cells of a dense cell: candidates from the 26 cells around (cx, cy, cz), filtered to
// those within `reach` of the cell, compacted into batches of 32.
template <bool WRAP>
__device__ __forceinline__ void tile_neighbours(const float4 *__restrict__ sorted,
                                                const unsigned int *__restrict__ cs, unsigned int *rel, float4 *s_pj,
                                                const float4 &me, int ib, int cntI, unsigned int grp, bool leader,
                                                int cx, int cy, int cz, const Grid &g, int lane,
                                                unsigned int &nedges, unsigned int &ntests)
{
    const int n = g.n;
    // lane q < 27 looks up neighbour cell q = (dx + 1) + 3 (dy + 1) + 9 (dz + 1); q > 13 is the forward half
    int nx = 0, ny = 0, nz = 0, beg = 0, len = 0;
    if (lane < 27 && lane != 13) {
        nx = cx + lane % 3 - 1;
        ny = cy + (lane / 3) % 3 - 1;
        nz = cz + lane / 9 - 1;
        if (WRAP) {
            nx = nx < 0 ? n - 1 : (nx >= n ? 0 : nx);
            ny = ny < 0 ? n - 1 : (ny >= n ? 0 : ny);
            nz = nz < 0 ? n - 1 : (nz >= n ? 0 : nz);
        }
        const unsigned int c = cell_id(nx, ny, nz, n);
        beg = (int)__ldg(cs + c);
        len = (int)__ldg(cs + c + 1) - beg;
        // a dense neighbour in my backward half owns our pairs itself
        if (len >= kDenseCell && lane < 13) len = 0;
    }
    int incl = len;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(kFull, incl, o);
        if (lane >= o) incl += v;
    }
    const int total = __shfl_sync(kFull, incl, 31);
    const int excl = incl - len;
    const float lo = g.reach, hi = 1.0f - g.reach;
    int nc = 0;  // candidates waiting in s_pj (warp-uniform)
    for (int base = 0; base < total; base += 32) {
        const int p = base + lane;
        const bool has = p < total;
        // owner q of slot p: the first lane whose inclusive prefix exceeds p
        int q = 0;
#pragma unroll
        for (int st = 16; st > 0; st >>= 1) {
            const int v = __shfl_sync(kFull, incl, q + st - 1);
            if (v <= p) q += st;
        }
        q = min(q, 31);
        const int j = __shfl_sync(kFull, beg, q) + (p - __shfl_sync(kFull, excl, q));
        const int qx = __shfl_sync(kFull, nx, q), qy = __shfl_sync(kFull, ny, q), qz = __shfl_sync(kFull, nz, q);
        bool pass = false;
        float4 pj = make_float4(0.f, 0.f, 0.f, 0.f);
        if (has) {
            pj = __ldg(sorted + j);
            // position of the candidate inside ITS cell; it can reach my cell only from within
            // `reach` of the face(s) it shares with it (the same margins as the sparse kernel's flags)
            const float fx = __fmul_rn(pj.x, g.inv_cell) - (float)qx;
            const float fy = __fmul_rn(pj.y, g.inv_cell) - (float)qy;
            const float fz = __fmul_rn(pj.z, g.inv_cell) - (float)qz;
            const int dx = q % 3 - 1, dy = (q / 3) % 3 - 1, dz = q / 9 - 1;
            pass = (dx == 0 || (dx < 0 ? fx > hi : fx < lo)) && (dy == 0 || (dy < 0 ? fy > hi : fy < lo)) &&
                   (dz == 0 || (dz < 0 ? fz > hi : fz < lo));
            pj.w = __int_as_float(j);
        }
        const unsigned int bal = __ballot_sync(kFull, pass);
        if (pass) s_pj[nc + __popc(bal & lanemask_lt())] = pj;
        nc += __popc(bal);
        __syncwarp();
        if (nc >= 32) {
            const unsigned int adjT = batch_adjacency<WRAP>(me, s_pj, 32, g, lane, nedges);
            ntests += 32u * (unsigned int)cntI;
            batch_unions(adjT, s_pj, 32, rel, ib, grp, leader, lane);
            const float4 keep = s_pj[32 + lane];
            __syncwarp();
            s_pj[lane] = keep;
            nc -= 32;
            __syncwarp();
        }
    }
    if (nc) {
        const unsigned int adjT = batch_adjacency<WRAP>(me, s_pj, nc, g, lane, nedges);
        ntests += (unsigned int)(nc * cntI);
        batch_unions(adjT, s_pj, nc, rel, ib, grp, leader, lane);
    }
    __syncwarp();
}

__global__ void __launch_bounds__(kLinkBlock) link_tiles_kernel(const float4 *__restrict__ sorted, Grid g,
                                                                const unsigned int *__restrict__ cell_start,
                                                                const unsigned long long *__restrict__ items,
                                                                unsigned int *rel, Ctrl *ctrl)
{
    __shared__ float4 s_pj_all[kWarpsPerCta][64];
    float4 *s_pj = s_pj_all[threadIdx.x >> 5];
    const int lane = threadIdx.x & 31;
    const unsigned int nitems = ctrl->ndense;
    const unsigned int nwarps = gridDim.x * kWarpsPerCta;
    const float inf = __int_as_float(0x7f800000);
    const int n = g.n;
    unsigned int nedges = 0, ntests = 0;  // warp-uniform
    for (unsigned int it = blockIdx.x * kWarpsPerCta + (threadIdx.x >> 5); it < nitems; it += nwarps) {
        const unsigned long long item = __ldg(items + it);
        const unsigned int c = (unsigned int)(item >> 32);
        const int t = (int)(unsigned int)item;
        const int b0 = (int)__ldg(cell_start + c), e0 = (int)__ldg(cell_start + c + 1);
        const int ts = (int)dense_tile_size((unsigned int)(e0 - b0));
        const int ib = b0 + t * ts;
        const int cntI = min(ts, e0 - ib);
        // a lane without a particle sits at +inf: d2 = inf (or NaN) fails every test
        float4 me = make_float4(inf, inf, inf, 0.0f);
        if (lane < cntI) me = __ldg(sorted + ib + lane);
        me.w = __int_as_float(ib + lane);

        // ---- the tile against itself (pairs inside one cell never wrap: cell side <= L/3)
        __syncwarp();
        s_pj[lane] = me;
        __syncwarp();
        unsigned int e_diag = 0;
        unsigned int adj = batch_adjacency<false>(me, s_pj, cntI, g, lane, e_diag) & ~(1u << lane);
        // every real particle is linked to itself (d2 = 0) and every pair shows up twice; a lane at
        // +inf gives inf - inf = NaN and is linked to nothing
        nedges += (e_diag - (unsigned int)cntI) >> 1;
        ntests += (unsigned int)(cntI * (cntI - 1) / 2);
        int lab = lane;  // lowest lane of my component inside the tile
        if (__any_sync(kFull, adj != 0u)) {
            // breadth-first from the lowest unlabelled lane; one warp OR-reduction per level
            const unsigned int self = 1u << lane;
            unsigned int todo = cntI >= 32 ? kFull : ((1u << cntI) - 1u);
            while (todo) {
                const int r = __ffs((int)todo) - 1;
                unsigned int vis = 1u << r;
                while (true) {
                    const unsigned int nxt = vis | __reduce_or_sync(kFull, (vis & self) ? adj : 0u);
                    if (nxt == vis) break;
                    vis = nxt;
                }
                if (vis & self) lab = r;
                todo &= ~vis;
            }
            if (lab != lane) unite_rel(rel, ib + lane, ib + lab);
        }
        const unsigned int grp = __match_any_sync(kFull, lab);
        const bool leader = lab == lane;

        // ---- the earlier tiles of my cell (all full: ts particles)
        for (int jt = 0; jt < t; ++jt) {
            const int jb = b0 + jt * ts;
            __syncwarp();
            if (lane < ts) {
                float4 pj = __ldg(sorted + jb + lane);
                pj.w = __int_as_float(jb + lane);
                s_pj[lane] = pj;
            }
            __syncwarp();
            const unsigned int adjT = batch_adjacency<false>(me, s_pj, ts, g, lane, nedges);
            ntests += (unsigned int)(ts * cntI);
            batch_unions(adjT, s_pj, ts, rel, ib, grp, leader, lane);
        }
        __syncwarp();

        // ---- the 26 neighbour cells
        const int cx = (int)(c % (unsigned int)n), cy = (int)((c / (unsigned int)n) % (unsigned int)n),
                  cz = (int)(c / ((unsigned int)n * (unsigned int)n));
        const bool wrap = n < 6 || cx == 0 || cx == n - 1 || cy == 0 || cy == n - 1 || cz == 0 || cz == n - 1;
        if (wrap) tile_neighbours<true>(sorted, cell_start, rel, s_pj, me, ib, cntI, grp, leader, cx, cy, cz, g, lane, nedges, ntests);
        else tile_neighbours<false>(sorted, cell_start, rel, s_pj, me, ib, cntI, grp, leader, cx, cy, cz, g, lane, nedges, ntests);
    }
    if (lane == 0) {
        if (nedges) atomicAdd(&ctrl->edges, (unsigned long long)nedges);
        if (ntests) atomicAdd(&ctrl->pair_tests, (unsigned long long)ntests);
    }
}

// =============================================================================================
// link_sparse_kernel: pairs of two sparse cells.
// =============================================================================================
constexpr int kStencil = 14;                        // own cell + 13 forward cells
constexpr int kMaxRanges = 32 * kStencil;           // candidate ranges of one warp
constexpr int kMaxSlots = kMaxRanges * (kDenseCell - 1);  // a sparse cell holds < kDenseCell particles
constexpr int kBitmapWords = (kMaxSlots + 31) / 32;

// Stencil order: q = 0 own cell, 1 the +x cell, then the rows (dy, dz) = (+1, 0), (-1, +1), (0, +1),
// (+1, +1) with dx = -1, 0, +1 each.
struct SparseSmem {
    int2 range[kMaxRanges];            // (first candidate, first slot << 5 | owner lane)
    unsigned int bitmap[kBitmapWords]; // bit p set: a range starts at slot p
};

template <bool WRAP>
__device__ __forceinline__ void sparse_warp(const float4 *__restrict__ sorted, const unsigned int *__restrict__ cs,
                                            unsigned int *rel, int si, bool valid, const float4 &me, int cx, int cy,
                                            int cz, float fx, float fy, float fz, const Grid &g, SparseSmem &sm,
                                            int lane, unsigned int &nedges, unsigned int &ntests)
{
    const int n = g.n;
    const float lo = g.reach, hi = 1.0f - g.reach;
    const bool xl = fx < lo, xh = fx > hi, yl = fy < lo, yh = fy > hi, zh = fz > hi;
    int beg[kStencil], len[kStencil];
    bool live = valid;
#pragma unroll
    for (int q = 0; q < kStencil; ++q) {
        const int dx = q == 0 ? 0 : (q == 1 ? 1 : (q - 2) % 3 - 1);
        const int dy = q < 2 ? 0 : (q < 5 ? 1 : (q < 8 ? -1 : (q < 11 ? 0 : 1)));
        const int dz = q < 5 ? 0 : 1;
        // the cell can hold a partner only if I am within `reach` of every face between us
        const bool want = live && (dx == 0 || (dx < 0 ? xl : xh)) && (dy == 0 || (dy < 0 ? yl : yh)) && (dz == 0 || zh);
        beg[q] = 0;
        len[q] = 0;
        if (want) {
            int ax = cx + dx, ay = cy + dy, az = cz + dz;
            if (WRAP) {
                ax = ax < 0 ? n - 1 : (ax >= n ? 0 : ax);
                ay = ay < 0 ? n - 1 : (ay >= n ? 0 : ay);
                az = az >= n ? 0 : az;
            }
            const unsigned int c = cell_id(ax, ay, az, n);
            const int b = (int)__ldg(cs + c), e = (int)__ldg(cs + c + 1);
            if (e - b < kDenseCell) {  // pairs with a dense cell belong to link_tiles_kernel
                beg[q] = q == 0 ? si + 1 : b;
                len[q] = e - beg[q];
            } else if (q == 0) {
                live = false;  // my own cell is dense: nothing to do here
            }
        }
    }
    // flatten: one packed warp scan gives every lane its first slot (low 16 bits) and range id (high)
    unsigned int mine = 0;
#pragma unroll
    for (int q = 0; q < kStencil; ++q) mine += (unsigned int)len[q] + (len[q] > 0 ? 0x10000u : 0u);
    unsigned int incl = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned int v = __shfl_up_sync(kFull, incl, o);
        if (lane >= o) incl += v;
    }
    const unsigned int all = __shfl_sync(kFull, incl, 31);
    const int total = (int)(all & 0xffffu);
    if (total == 0) return;
    const int words = (total + 31) >> 5;
    for (int w = lane; w < words; w += 32) sm.bitmap[w] = 0u;
    __syncwarp();
    {
        int slot = (int)((incl - mine) & 0xffffu), rid = (int)((incl - mine) >> 16);
#pragma unroll
        for (int q = 0; q < kStencil; ++q)
            if (len[q] > 0) {
                sm.range[rid++] = make_int2(beg[q], (slot << 5) | lane);
                atomicOr(&sm.bitmap[slot >> 5], 1u << (slot & 31));
                slot += len[q];
            }
    }
    __syncwarp();
    if (lane == 0) ntests += (unsigned int)total;
    const unsigned int le = lanemask_lt() | (1u << lane);
    int before = 0;  // ranges that start in earlier words
    for (int w = 0; w < words; ++w) {
        const unsigned int bits = sm.bitmap[w];
        const int p = (w << 5) + lane;
        const int2 r = sm.range[before + __popc(bits & le) - 1];  // p >= 0 has a range: slot 0 starts one
        before += __popc(bits);
        const int owner = r.y & 31;
        float4 o4;
        o4.x = __shfl_sync(kFull, me.x, owner);
        o4.y = __shfl_sync(kFull, me.y, owner);
        o4.z = __shfl_sync(kFull, me.z, owner);
        o4.w = 0.0f;
        const int osi = __shfl_sync(kFull, si, owner);
        if (p < total) {
            const int j = r.x + (p - (r.y >> 5));
            const float4 pj = __ldg(sorted + j);
            if (linked_t<WRAP>(o4, pj, g)) {
                ++nedges;
                unite_rel(rel, osi, j);
            }
        }
    }
    __syncwarp();
}

// Persistent grid: each warp walks chunks of 32 consecutive cell-sorted particles.
__global__ void __launch_bounds__(kLinkBlock) link_sparse_kernel(const float4 *__restrict__ sorted, int64_t N, Grid g,
                                                                 const unsigned int *__restrict__ cell_start,
                                                                 unsigned int *rel, Ctrl *ctrl)
{
    __shared__ SparseSmem s_all[kWarpsPerCta];
    SparseSmem &sm = s_all[threadIdx.x >> 5];
    const int lane = threadIdx.x & 31;
    unsigned int nedges = 0, ntests = 0;  // per lane
    const int n = g.n;
    const float lo = g.reach, hi = 1.0f - g.reach;
    for (int64_t base = (int64_t)blockIdx.x * kLinkBlock; base < N; base += (int64_t)gridDim.x * kLinkBlock) {
        const int64_t s64 = base + threadIdx.x;
        const bool valid = s64 < N;
        const int si = (int)s64;
        float4 me = make_float4(0.f, 0.f, 0.f, 0.f);
        int cx = 0, cy = 0, cz = 0;
        float fx = 0.5f, fy = 0.5f, fz = 0.5f;
        bool needwrap = false;
        if (valid) {
            me = __ldg(sorted + si);
            const float ux = __fmul_rn(me.x, g.inv_cell), uy = __fmul_rn(me.y, g.inv_cell),
                        uz = __fmul_rn(me.z, g.inv_cell);
            cx = min(__float2int_rd(ux), g.n_minus_1);
            cy = min(__float2int_rd(uy), g.n_minus_1);
            cz = min(__float2int_rd(uz), g.n_minus_1);
            fx = ux - (float)cx;
            fy = uy - (float)cy;
            fz = uz - (float)cz;
            needwrap = n < 6 || (fx < lo && cx == 0) || (fx > hi && cx == n - 1) || (fy < lo && cy == 0) ||
                       (fy > hi && cy == n - 1) || (fz > hi && cz == n - 1);
        }
        if (__any_sync(kFull, needwrap))
            sparse_warp<true>(sorted, cell_start, rel, si, valid, me, cx, cy, cz, fx, fy, fz, g, sm, lane, nedges, ntests);
        else
            sparse_warp<false>(sorted, cell_start, rel, si, valid, me, cx, cy, cz, fx, fy, fz, g, sm, lane, nedges, ntests);
    }
    for (int o = 16; o > 0; o >>= 1) {
        nedges += __shfl_xor_sync(kFull, nedges, o);
        ntests += __shfl_xor_sync(kFull, ntests, o);
    }
    if (lane == 0) {  // one pair of global atomics per warp: no CTA barrier at the end
        if (nedges) atomicAdd(&ctrl->edges, (unsigned long long)nedges);
        if (ntests) atomicAdd(&ctrl->pair_tests, (unsigned long long)ntests);
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
                        const unsigned long long *dense_list, unsigned int *rel, Ctrl *ctrl, int num_sms,
                        cudaStream_t s)
{
    if (N <= 0) return cudaSuccess;
    const unsigned int grid = (unsigned int)min((int64_t)blocks_for(N, kLinkBlock), (int64_t)num_sms * 32);
    link_tiles_kernel<<<(unsigned int)num_sms * 8, kLinkBlock, 0, s>>>(sorted, g, cell_start, dense_list, rel, ctrl);
    link_sparse_kernel<<<grid, kLinkBlock, 0, s>>>(sorted, N, g, cell_start, rel, ctrl);
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
