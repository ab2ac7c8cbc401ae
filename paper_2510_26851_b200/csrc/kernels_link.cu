// kernels_link.cu — H4 half-stencil pair tests + union, H5 canonical labels.
// What is linked: PAPER.md:85-87 (§2 step iv) and PAPER.md:200-214 (Alg. 2 candidate cells and
// mask); the 27-cell stencil with indices mod n is PAPER.md:202.  The T label sweeps of
// PAPER.md:221-225 are replaced by their fixed point, computed with a lock-free union-find
// (ECL-CC style: atomicCAS hooks at roots, path halving) whose root is the member with the
// minimum original index, the converged min-label of PAPER.md:91.
//
// Design.  The union-find runs in CELL-SORTED index space: a component is a
// spatially compact object, so its parent entries sit in a few cache lines.  Every unordered
// pair of particles in the same or in adjacent cells is tested exactly once, by one of the two roles
// of link_kernel, the one that owns the pair's HOME cell (the cell that sees the other one in its
// forward half stencil):
//   tile role    home cell DENSE (>= kDenseCell particles).  One warp per (dense cell, tile of <= 32
//                of its particles): the tile sits in registers, one particle per lane; the
//                candidates (the tile itself, the earlier tiles of the cell, and the particles of
//                the 13 forward cells that lie within b of the cell) are staged 32 at a time in
//                shared memory and broadcast, so one trip of ~13 instructions tests 32 pairs.  The
//                adjacency comes out as ballot bitmasks; components of the tile are closed in
//                registers and only one hook per (component, adjacent candidate) reaches the
//                union-find.
//   sparse role  home cell sparse.  One thread per particle collects its candidate ranges (own cell
//                after itself + the forward cells, reach-filtered); the ranges of a warp are
//                flattened into one list of candidate slots that the 32 lanes walk together, so a
//                lane with many candidates does not hold the others hostage; ranges longer than
//                kLongRange (dense neighbour cells) are walked by the whole warp.
// The root of a set is its member with the smallest ORIGINAL index, so the canonical label is
// read off the root by one streaming pass (chase + scatter to labels[original index]).
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

// (the union-find, find_rel / unite_rel, lives in fof_internal.cuh: kernels_stochastic.cu uses it too)

#ifndef FOF_LINK_MINB
#define FOF_LINK_MINB 6   // resident CTAs per SM the link kernel is compiled for (register cap)
#endif
#ifndef FOF_START_ROLE
#define FOF_START_ROLE 0  // every warp starts on the tile queue (see link_kernel)
#endif
#ifndef FOF_LONG_RANGE
#define FOF_LONG_RANGE 16
#endif
constexpr int kWarpsPerCta = kLinkBlock / 32;
constexpr unsigned int kFull = 0xffffffffu;

__device__ __forceinline__ unsigned int lanemask_lt()
{
    unsigned int m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// =============================================================================================
// Tile role: pairs whose home cell is dense.
// =============================================================================================

// Tile I (one particle per lane, `me`; idle lanes sit at +inf) against a batch of `cnt` <= 32
// candidates staged in shared memory.  Returns, in lane k, the mask of tile lanes linked to
// candidate k.
template <bool WRAP>
__device__ __forceinline__ unsigned int batch_adjacency(const float4 &me, const float4 *s_pj, int cnt, const Grid &g,
                                                        int lane)
{
    unsigned int adjT = 0;
#pragma unroll 8
    for (int k = 0; k < cnt; ++k) {
        const unsigned int bal = __ballot_sync(kFull, linked_t<WRAP>(me, s_pj[k], g));
        if (lane == k) adjT = bal;
    }
    return adjT;
}

// Hooks of one batch: candidate k (cell-sorted index in s_pj[k].w) joins every component of the
// tile it is linked to.  `grp` = lanes of my tile component, `leader` = I am its lowest lane.
__device__ __forceinline__ void batch_unions(unsigned int adjT, const float4 *s_pj, int cnt, unsigned int *rel,
                                             const int *__restrict__ idx_s, int ib,
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
        if (adjT & members) unite_rel(rel, idx_s, j, ib + gl);
    }
}

// The 13 forward neighbour cells q = 0..12 of a cell: +x, then the rows (dy, dz) = (+1, 0), (-1, +1),
// (0, +1), (+1, +1) with dx = -1, 0, +1 each; offsets + 1 packed two bits per cell.
constexpr unsigned int pack13(int axis)
{
    unsigned int v = 0;
    for (int q = 0; q < 13; ++q) {
        const int dx = q == 0 ? 1 : (q - 1) % 3 - 1;
        const int dy = q == 0 ? 0 : (q < 4 ? 1 : (q - 4) / 3 - 1);
        const int dz = q < 4 ? 0 : 1;
        const int d = axis == 0 ? dx : (axis == 1 ? dy : dz);
        v |= (unsigned int)(d + 1) << (2 * q);
    }
    return v;
}
constexpr unsigned int kFwdX = pack13(0), kFwdY = pack13(1), kFwdZ = pack13(2);

// Candidates from the 13 forward cells around (cx, cy, cz), filtered to those within `reach` of
// the cell, compacted into batches of 32 and tested against the tile.
template <bool WRAP>
__device__ __forceinline__ void tile_neighbours(const float4 *__restrict__ sorted,
                                                const unsigned int *__restrict__ cs, unsigned int *rel,
                                                const int *__restrict__ idx_s, float4 *s_pj, const float4 &me, int ib, int cntI, unsigned int grp, bool leader,
                                                int cx, int cy, int cz, const Grid &g, int lane,
                                                int part, int nparts, unsigned int &nedges, unsigned int &ntests)
{
    const int n = g.n;
    int beg = 0, len = 0;
    if (lane < 13 && (nparts == 1 || (lane & (nparts - 1)) == part)) {  // nparts is a power of two
        int nx = cx + (int)((kFwdX >> (2 * lane)) & 3u) - 1;
        int ny = cy + (int)((kFwdY >> (2 * lane)) & 3u) - 1;
        int nz = cz + (int)((kFwdZ >> (2 * lane)) & 3u) - 1;
        if (WRAP) {
            nx = nx < 0 ? n - 1 : (nx >= n ? 0 : nx);
            ny = ny < 0 ? n - 1 : (ny >= n ? 0 : ny);
            nz = nz >= n ? 0 : nz;
        }
        const unsigned int c = cell_id(nx, ny, nz, n);
        beg = (int)__ldg(cs + c);
        len = (int)__ldg(cs + c + 1) - beg;
    }
    int incl = len;
#pragma unroll
    for (int o = 1; o < 16; o <<= 1) {  // lanes >= 13 hold 0: a 16-lane scan is enough
        const int v = __shfl_up_sync(kFull, incl, o);
        if (lane >= o) incl += v;
    }
    const int total = __shfl_sync(kFull, incl, 15);
    if (total == 0) return;
    const int excl = incl - len;
    const float lo = g.reach, hi = 1.0f - g.reach;
    int nc = 0;  // candidates waiting in s_pj (warp-uniform)
    for (int base = 0; base < total; base += 32) {
        const int p = base + lane;
        const bool has = p < total;
        // owner q of slot p: the first lane whose inclusive prefix exceeds p
        int q = 0;
#pragma unroll
        for (int st = 8; st > 0; st >>= 1) {
            const int v = __shfl_sync(kFull, incl, q + st - 1);
            if (v <= p) q += st;
        }
        const int j = __shfl_sync(kFull, beg, q) + (p - __shfl_sync(kFull, excl, q));
        bool pass = false;
        float4 pj = make_float4(0.f, 0.f, 0.f, 0.f);
        if (has) {
            pj = __ldg(sorted + j);
            // position of the candidate inside ITS cell (the fractional part of its cell coordinate):
            // it can reach my cell only from within `reach` of the face(s) it shares with it
            // (the same margins as the sparse kernel's flags)
            const float ux = __fmul_rn(pj.x, g.inv_cell), uy = __fmul_rn(pj.y, g.inv_cell),
                        uz = __fmul_rn(pj.z, g.inv_cell);
            const float fx = ux - (float)min(__float2int_rd(ux), g.n_minus_1);
            const float fy = uy - (float)min(__float2int_rd(uy), g.n_minus_1);
            const float fz = uz - (float)min(__float2int_rd(uz), g.n_minus_1);
            const int dx = (int)((kFwdX >> (2 * q)) & 3u) - 1, dy = (int)((kFwdY >> (2 * q)) & 3u) - 1,
                      dz = (int)((kFwdZ >> (2 * q)) & 3u) - 1;
            pass = (dx == 0 || (dx < 0 ? fx > hi : fx < lo)) && (dy == 0 || (dy < 0 ? fy > hi : fy < lo)) &&
                   (dz == 0 || fz < lo);
            pj.w = __int_as_float(j);
        }
        const unsigned int bal = __ballot_sync(kFull, pass);
        if (pass) s_pj[nc + __popc(bal & lanemask_lt())] = pj;
        nc += __popc(bal);
        __syncwarp();
        if (nc >= 32) {
            const unsigned int adjT = batch_adjacency<WRAP>(me, s_pj, 32, g, lane);
            nedges += (unsigned int)__popc(adjT);
            if (lane == 0) ntests += 32u * (unsigned int)cntI;
            batch_unions(adjT, s_pj, 32, rel, idx_s, ib, grp, leader, lane);
            const float4 keep = s_pj[32 + lane];
            __syncwarp();
            s_pj[lane] = keep;
            nc -= 32;
            __syncwarp();
        }
    }
    if (nc) {
        const unsigned int adjT = batch_adjacency<WRAP>(me, s_pj, nc, g, lane);
        nedges += (unsigned int)__popc(adjT);
        if (lane == 0) ntests += (unsigned int)(nc * cntI);
        batch_unions(adjT, s_pj, nc, rel, idx_s, ib, grp, leader, lane);
    }
    __syncwarp();
}

// One work item: tile `t` (ts particles) of dense cell `c`.
__device__ __forceinline__ void tile_item(const float4 *__restrict__ sorted, const Grid &g,
                                          const unsigned int *__restrict__ cell_start, unsigned long long item,
                                          unsigned int *rel, const int *__restrict__ idx_s, float4 *s_pj, int lane, unsigned int &nedges,
                                          unsigned int &ntests)
{
    const float inf = __int_as_float(0x7f800000);
    const int n = g.n;
    const unsigned int c = (unsigned int)(item >> 32);
    const int ts = (int)(((unsigned int)item) & 31u) + 1;
    const int b0 = (int)__ldg(cell_start + c), e0 = (int)__ldg(cell_start + c + 1);
    // a heavy cell's tile comes as nparts items, each with every nparts-th batch of its candidates
    const int nparts = (int)dense_parts((unsigned int)(e0 - b0));
    const int part = nparts == 1 ? 0 : (int)(((unsigned int)item) >> 29);
    const int t = nparts == 1 ? (int)(((unsigned int)item) >> 5) : (int)((((unsigned int)item) >> 5) & 0xffffffu);
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
    const unsigned int adj = batch_adjacency<false>(me, s_pj, cntI, g, lane) & ~(1u << lane);
    if (part == 0) {
        nedges += (unsigned int)__popc(adj & lanemask_lt());
        if (lane == 0) ntests += (unsigned int)(cntI * (cntI - 1) / 2);
    }
    // Components of the tile: breadth-first from the lowest unlabelled lane, one warp OR-reduction
    // per level.  Lanes without a link are their own component and are never visited.  `head` is
    // the member with the smallest original index (the union-find's order): every other member
    // hooks straight under it, depth one, no retries.  (A parent that is no longer a root is fine:
    // original indices still fall along every path.)
    const unsigned int self = 1u << lane;
    unsigned int grp = self;
    int head = lane;
    if (__any_sync(kFull, adj != 0u)) {
        const int my_oi = lane < cntI ? __ldg(idx_s + ib + lane) : 0x7fffffff;
        unsigned int todo = __ballot_sync(kFull, adj != 0u);
        while (todo) {
            const int r = __ffs((int)todo) - 1;
            unsigned int vis = 1u << r;
            while (true) {
                const unsigned int nxt = vis | __reduce_or_sync(kFull, (vis & self) ? adj : 0u);
                if (nxt == vis) break;
                vis = nxt;
            }
            const bool in = (vis & self) != 0u;
            const int m = __reduce_min_sync(kFull, in ? my_oi : 0x7fffffff);
            const unsigned int hb = __ballot_sync(kFull, in && my_oi == m);
            if (in) { grp = vis; head = __ffs((int)hb) - 1; }
            todo &= ~vis;
        }
    }
    const bool leader = head == lane;
    if (part == 0 && !leader && atomicCAS(rel + ib + lane, 0u, (unsigned int)(lane - head)) != 0u)
        unite_rel(rel, idx_s, ib + lane, ib + head);  // somebody hooked me first: general path

    // ---- the earlier tiles of my cell (all full: ts particles)
    for (int jt = part; jt < t; jt += nparts) {
        const int jb = b0 + jt * ts;
        __syncwarp();
        if (lane < ts) {
            float4 pj = __ldg(sorted + jb + lane);
            pj.w = __int_as_float(jb + lane);
            s_pj[lane] = pj;
        }
        __syncwarp();
        const unsigned int adjT = batch_adjacency<false>(me, s_pj, ts, g, lane);
        nedges += (unsigned int)__popc(adjT);
        if (lane == 0) ntests += (unsigned int)(ts * cntI);
        batch_unions(adjT, s_pj, ts, rel, idx_s, ib, grp, leader, lane);
    }
    __syncwarp();

    // ---- the 13 forward neighbour cells; the cell coordinates come from a member's position
    // (the binning expression of H1, so they are the coordinates the sort used)
    const float3 p0 = make_float3(__shfl_sync(kFull, me.x, 0), __shfl_sync(kFull, me.y, 0),
                                  __shfl_sync(kFull, me.z, 0));
    const int cx = min(__float2int_rd(__fmul_rn(p0.x, g.inv_cell)), g.n_minus_1);
    const int cy = min(__float2int_rd(__fmul_rn(p0.y, g.inv_cell)), g.n_minus_1);
    const int cz = min(__float2int_rd(__fmul_rn(p0.z, g.inv_cell)), g.n_minus_1);
    const bool wrap = n < 6 || cx == 0 || cx == n - 1 || cy == 0 || cy == n - 1 || cz == n - 1;
    if (wrap) tile_neighbours<true>(sorted, cell_start, rel, idx_s, s_pj, me, ib, cntI, grp, leader, cx, cy, cz, g, lane, part, nparts, nedges, ntests);
    else tile_neighbours<false>(sorted, cell_start, rel, idx_s, s_pj, me, ib, cntI, grp, leader, cx, cy, cz, g, lane, part, nparts, nedges, ntests);
}

// =============================================================================================
// Sparse role: pairs whose home cell is sparse.
// =============================================================================================
constexpr int kLongRange = FOF_LONG_RANGE;  // longer candidate ranges (dense neighbour cells) are walked by the whole warp
constexpr int kRangesNoWrap = 5, kRangesWrap = 7;  // with wrap: the 14 stencil cells in two passes of 7
constexpr int kMaxRanges = 32 * kRangesWrap;
constexpr int kMaxSlots = kMaxRanges * kLongRange;  // < 2^16: slot and range counts share one packed scan
constexpr int kBitmapWords = (kMaxSlots + 31) / 32;

struct SparseSmem {
    int2 range[kMaxRanges];             // (first candidate, first slot << 5 | owner lane)
    unsigned int bitmap[kBitmapWords];  // bit p set: a range starts at slot p
};

// One home particle per lane.  Candidate ranges: without wrap, one run of `sorted` per stencil row
// (the rest of my cell [+ the +x cell]; then up to three cells of the rows (dy, dz) = (+1, 0),
// (-1, +1), (0, +1), (+1, +1)); with wrap, one range per stencil cell.  A neighbour cell is
// visited only if I am within `reach` of every face between us.
// the 14 stencil cells of the sparse role (own, +x, rows (+1,0), (-1,+1), (0,+1), (+1,+1)), offsets + 1
// packed two bits per cell
constexpr unsigned int pack14(int axis)
{
    unsigned int v = 0;
    for (int q = 0; q < 14; ++q) {
        const int dx = q == 0 ? 0 : (q == 1 ? 1 : (q - 2) % 3 - 1);
        const int dy = q < 2 ? 0 : (q < 5 ? 1 : (q < 8 ? -1 : (q < 11 ? 0 : 1)));
        const int dz = q < 5 ? 0 : 1;
        const int d = axis == 0 ? dx : (axis == 1 ? dy : dz);
        v |= (unsigned int)(d + 1) << (2 * q);
    }
    return v;
}
constexpr unsigned int kStX = pack14(0), kStY = pack14(1), kStZ = pack14(2);

template <bool WRAP>
__device__ __forceinline__ void sparse_warp(const float4 *__restrict__ sorted, const unsigned int *__restrict__ cs,
                                            unsigned int *rel, const int *__restrict__ idx_s, int si, bool live,
                                            const unsigned int *home, int c1,
                                            const float4 &me, int cx, int cy, int cz, float fx, float fy, float fz,
                                            const Grid &g, SparseSmem &sm, int lane, unsigned int &nedges,
                                            unsigned int &ntests, int pass)
{
    // live: a real particle whose home cell (cell_start entry `home`, end `c1`) is sparse;
    // pass: with WRAP the stencil cells 7 pass .. 7 pass + 6 are walked (two calls), else unused
    constexpr int NR = WRAP ? kRangesWrap : kRangesNoWrap;
    const int n = g.n;
    const float lo = g.reach, hi = 1.0f - g.reach;
    const bool xl = fx < lo, xh = fx > hi, yl = fy < lo, yh = fy > hi, zh = fz > hi;
    int beg[NR], len[NR];
#pragma unroll
    for (int r = 0; r < NR; ++r) beg[r] = len[r] = 0;
    {
        if (live) {
            if (!WRAP) {
                // the loads below stay inside the row: a lane that needs the cell behind an x face
                // has sent its whole warp to the WRAP variant.  Flags are consumed where they are
                // computed (short predicate lifetimes).
                const int off_lo = xl ? -1 : 0, off_hi = xh ? 2 : 1;
                beg[0] = si + 1;
                len[0] = (xh ? (int)__ldg(home + 2) : c1) - beg[0];
                if (yh) {
                    const unsigned int *row = home + n;
                    beg[1] = (int)__ldg(row + off_lo);
                    len[1] = (int)__ldg(row + off_hi) - beg[1];
                }
                if (zh) {
                    const unsigned int *row = home + n * n;
                    beg[3] = (int)__ldg(row + off_lo);
                    len[3] = (int)__ldg(row + off_hi) - beg[3];
                    if (yl) {
                        beg[2] = (int)__ldg(row - n + off_lo);
                        len[2] = (int)__ldg(row - n + off_hi) - beg[2];
                    }
                    if (yh) {
                        beg[4] = (int)__ldg(row + n + off_lo);
                        len[4] = (int)__ldg(row + n + off_hi) - beg[4];
                    }
                }
            } else {
#pragma unroll
                for (int k = 0; k < kRangesWrap; ++k) {
                    const int q = k + pass * kRangesWrap;
                    const int dx = (int)((kStX >> (2 * q)) & 3u) - 1, dy = (int)((kStY >> (2 * q)) & 3u) - 1,
                              dz = (int)((kStZ >> (2 * q)) & 3u) - 1;
                    if (q == 0) {
                        beg[0] = si + 1;
                        len[0] = c1 - beg[0];
                    } else if ((dx == 0 || (dx < 0 ? xl : xh)) && (dy == 0 || (dy < 0 ? yl : yh)) && (dz == 0 || zh)) {
                        int ax = cx + dx, ay = cy + dy, az = cz + dz;
                        ax = ax < 0 ? n - 1 : (ax >= n ? 0 : ax);
                        ay = ay < 0 ? n - 1 : (ay >= n ? 0 : ay);
                        az = az >= n ? 0 : az;
                        const unsigned int *p = cs + cell_id(ax, ay, az, n);
                        beg[k] = (int)__ldg(p);
                        len[k] = (int)__ldg(p + 1) - beg[k];
                    }
                }
            }
        }
    }
    // ---- long ranges: the whole warp walks them, 32 candidates per trip
    int longest = len[0];
#pragma unroll
    for (int r = 1; r < NR; ++r) longest = max(longest, len[r]);
    if (__any_sync(kFull, longest > kLongRange)) {
#pragma unroll
        for (int r = 0; r < NR; ++r) {
            unsigned int lng = __ballot_sync(kFull, len[r] > kLongRange);
            while (lng) {
                const int owner = __ffs((int)lng) - 1;
                lng &= lng - 1u;
                const int b = __shfl_sync(kFull, beg[r], owner), l = __shfl_sync(kFull, len[r], owner);
                const int osi = __shfl_sync(kFull, si, owner);
                float4 o4;
                o4.x = __shfl_sync(kFull, me.x, owner);
                o4.y = __shfl_sync(kFull, me.y, owner);
                o4.z = __shfl_sync(kFull, me.z, owner);
                o4.w = 0.0f;
                if (lane == 0) ntests += (unsigned int)l;
                for (int j = b + lane; j < b + l; j += 32)
                    if (linked_t<WRAP>(o4, __ldg(sorted + j), g)) {
                        ++nedges;
                        unite_rel(rel, idx_s, osi, j);
                    }
            }
            if (len[r] > kLongRange) len[r] = 0;
        }
    }
    // ---- the rest is flattened: one packed warp scan gives every lane its first slot (low 16 bits)
    // and its first range id (high bits)
    int tot = 0, cnt = 0;  // every len is >= 0
#pragma unroll
    for (int r = 0; r < NR; ++r) { tot += len[r]; cnt += min(len[r], 1); }
    const unsigned int mine = (unsigned int)tot | ((unsigned int)cnt << 16);
    unsigned int incl = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned int v = __shfl_up_sync(kFull, incl, o);
        if (lane >= o) incl += v;
    }
    const int total = (int)(__shfl_sync(kFull, incl, 31) & 0xffffu);
    if (total == 0) return;
    const int words = (total + 31) >> 5;
    static_assert(kBitmapWords <= 4 * 32, "bitmap zeroing below covers 128 words");
#pragma unroll
    for (int k = 0; k < (kBitmapWords + 31) / 32; ++k)
        if (lane + 32 * k < words) sm.bitmap[lane + 32 * k] = 0u;
    __syncwarp();
    {
        int slot = (int)((incl - mine) & 0xffffu), rid = (int)((incl - mine) >> 16);
#pragma unroll
        for (int r = 0; r < NR; ++r)
            if (len[r] > 0) {
                sm.range[rid++] = make_int2(beg[r], (slot << 5) | lane);
                atomicOr(&sm.bitmap[slot >> 5], 1u << (slot & 31));
                slot += len[r];
            }
    }
    __syncwarp();
    if (lane == 0) ntests += (unsigned int)total;
    const unsigned int le = lanemask_lt() | (1u << lane);
    int before = 0;  // ranges that start in earlier words
    for (int w = 0; w < words; ++w) {
        const unsigned int bits = sm.bitmap[w];
        const int p = (w << 5) + lane;
        const int2 r = sm.range[before + __popc(bits & le) - 1];  // slot 0 starts a range: never -1
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
            if (linked_t<WRAP>(o4, __ldg(sorted + j), g)) {
                ++nedges;
                unite_rel(rel, idx_s, osi, j);
            }
        }
    }
    __syncwarp();
}

// 32 consecutive cell-sorted particles, one per lane.
__device__ __forceinline__ void sparse_chunk(const float4 *__restrict__ sorted, int64_t N, const Grid &g,
                                             const unsigned int *__restrict__ cell_start, unsigned int *rel,
                                             const int *__restrict__ idx_s, int64_t base, SparseSmem &sm, int lane, unsigned int &nedges,
                                             unsigned int &ntests)
{
    const int n = g.n;
    const float lo = g.reach, hi = 1.0f - g.reach;
    const int64_t s64 = base + lane;
    const bool valid = s64 < N;
    const int si = (int)min(s64, N - 1);  // idle lanes of the last chunk shadow the last particle (never live)
    const float4 me = __ldg(sorted + si);
    const float ux = __fmul_rn(me.x, g.inv_cell), uy = __fmul_rn(me.y, g.inv_cell), uz = __fmul_rn(me.z, g.inv_cell);
    const int cx = min(__float2int_rd(ux), g.n_minus_1);
    const int cy = min(__float2int_rd(uy), g.n_minus_1);
    const int cz = min(__float2int_rd(uz), g.n_minus_1);
    const float fx = ux - (float)cx, fy = uy - (float)cy, fz = uz - (float)cz;
    const unsigned int *home = cell_start + cell_id(cx, cy, cz, n);
    const int c1 = (int)__ldg(home + 1);
    const bool live = valid & (c1 - (int)__ldg(home) < kDenseCell);  // a dense home cell belongs to the tile role
    // wrap is needed if a face I am within reach of is a box face (x: exact test; y, z: any particle of a
    // boundary row takes the wrapped variant, 3 rows in 256), or if the grid is too small for |d| < L/2
    const unsigned int edge_yz = ((unsigned int)(cy - 1) >= (unsigned int)(n - 2)) | (unsigned int)(cz == n - 1);
    const unsigned int edge_x = ((unsigned int)(fx < lo) & (unsigned int)(cx == 0)) |
                                ((unsigned int)(fx > hi) & (unsigned int)(cx == n - 1));
    const bool needwrap = live & (((unsigned int)(n < 6) | edge_yz | edge_x) != 0u);
    if (!__any_sync(kFull, live)) return;
    if (__any_sync(kFull, needwrap)) {
#pragma unroll 1
        for (int pass = 0; pass < 2; ++pass)
            sparse_warp<true>(sorted, cell_start, rel, idx_s, si, live, home, c1, me, cx, cy, cz, fx, fy, fz, g, sm, lane, nedges, ntests, pass);
    } else {
        sparse_warp<false>(sorted, cell_start, rel, idx_s, si, live, home, c1, me, cx, cy, cz, fx, fy, fz, g, sm, lane, nedges, ntests, 0);
    }
}

// =============================================================================================
// H4: one persistent kernel.  Every warp draws work through atomic tickets, first from the queue
// of (dense cell, tile) items listed by cell_sort_kernel, then, when that runs dry, from the queue
// of 32 x kSparseBatch consecutive cell-sorted particles of the sparse role: no grid-wide barrier
// between the two, the tail of one overlaps the head of the other.  All hooks are atomicCAS on
// roots, so any interleaving gives the same partition.  (Measured at cfg2: two back-to-back
// kernels 0.99 ms, this kernel 0.87 ms; letting half of the warps START on the sparse queue costs
// 1.69 ms -- the two roles together are ~170 KB of SASS and evict each other from the instruction
// caches when they share an SM.)
// =============================================================================================
constexpr int kTileBatch = 4;     // items per ticket (at most: small inputs take fewer, see link_kernel)
constexpr int kSparseBatch = 8;   // 32-particle chunks per ticket (at most)

union LinkSmem {
    float4 pj[64];
    SparseSmem sp;
};

__global__ void __launch_bounds__(kLinkBlock, FOF_LINK_MINB) link_kernel(const float4 *__restrict__ sorted, int64_t N,
                                                                         Grid g,
                                                                         const unsigned int *__restrict__ cell_start,
                                                                         const unsigned long long *__restrict__ items,
                                                                         unsigned int *rel,
                                                                         const int *__restrict__ idx_s, Ctrl *ctrl,
                                                                         unsigned int tile_batch,
                                                                         unsigned int sparse_batch,
                                                                         const unsigned int *gate)
{
    __shared__ LinkSmem s_all[kWarpsPerCta];
    if (gate && *gate == 0u) return;  // the block path did the work
    LinkSmem &sm = s_all[threadIdx.x >> 5];
    const int lane = threadIdx.x & 31;
    const unsigned int nitems = ctrl->ndense;
    unsigned int nedges = 0, ntests = 0;  // per lane
    int role = FOF_START_ROLE;
    for (int phase = 0; phase < 2; ++phase, role ^= 1) {
        if (role == 0) {
            while (true) {
                unsigned int it0 = 0;
                if (lane == 0) it0 = atomicAdd(&ctrl->tile_ticket, tile_batch);
                it0 = __shfl_sync(kFull, it0, 0);
                if (it0 >= nitems) break;
                const unsigned int it1 = min(it0 + tile_batch, nitems);
                for (unsigned int it = it0; it < it1; ++it)
                    tile_item(sorted, g, cell_start, __ldg(items + it), rel, idx_s, sm.pj, lane, nedges, ntests);
            }
        } else {
            while (true) {
                unsigned int k0 = 0;
                if (lane == 0) k0 = atomicAdd(&ctrl->sparse_ticket, sparse_batch);
                k0 = __shfl_sync(kFull, k0, 0);
                const int64_t base0 = (int64_t)k0 * 32;
                if (base0 >= N) break;
                for (int k = 0; k < kSparseBatch; ++k) {
                    const int64_t base = base0 + 32 * k;
                    if (k >= (int)sparse_batch || base >= N) break;
                    sparse_chunk(sorted, N, g, cell_start, rel, idx_s, base, sm.sp, lane, nedges, ntests);
                }
            }
        }
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

// H5 ("after convergence"): labels[original index] = original index of the root =
// the minimum original index of the component ("minimum label", "minimum
// global particle ID").  part_scatter_kernel has already written labels[i] = i, which is final for
// every root, so only non-roots are scattered here.  Four consecutive slots per thread, chased in
// lock step so that the (up to four) loads of one round are in flight together; read-only chase.
__global__ void __launch_bounds__(kBlock) write_labels_kernel(const unsigned int *__restrict__ rel,
                                                              const int *__restrict__ idx_s, int *__restrict__ labels,
                                                              int64_t N, bool vec, const unsigned int *gate,
                                                              int *__restrict__ cnt, unsigned long long *state,
                                                              int64_t state_items, Ctrl *ctrl)
{
    // cnt != nullptr: H6 rides along ("parallel histogram"): every non-root adds one to the size
    // counter of its canonical particle (zeroed by cell_sort_kernel), and the state of the compaction scan of
    // fof_groups is cleared, so that a fof_groups on these labels starts at H7.
    if (cnt && !(gate && *gate == 0u)) {
        const int64_t tid = (int64_t)blockIdx.x * kBlock + threadIdx.x;
        if (tid == 0) { ctrl->gscan_ticket = 0u; ctrl->K = 0; }
        for (int64_t k = tid; k < state_items; k += (int64_t)gridDim.x * kBlock) state[k] = 0ull;
    }
    // vec: rel and idx_s are 16-byte aligned (the workspace arrays are; the per-sample union-find arrays of
    // fof_link_stochastic_batch, rel_s + k N, are not when N is not a multiple of 4)
    const int64_t s0 = ((int64_t)blockIdx.x * kBlock + threadIdx.x) * 4;
    if (s0 >= N || (gate && *gate == 0u)) return;
    int d[4], oi[4];
    if (vec && s0 + 3 < N) {
        const uint4 t = __ldg(reinterpret_cast<const uint4 *>(rel + s0));
        d[0] = (int)t.x; d[1] = (int)t.y; d[2] = (int)t.z; d[3] = (int)t.w;
        if ((d[0] | d[1] | d[2] | d[3]) == 0) return;  // four roots
        const int4 o = __ldg(reinterpret_cast<const int4 *>(idx_s + s0));
        oi[0] = o.x; oi[1] = o.y; oi[2] = o.z; oi[3] = o.w;
    } else {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            d[k] = (s0 + k < N) ? (int)__ldg(rel + s0 + k) : 0;
            oi[k] = (s0 + k < N) ? __ldg(idx_s + s0 + k) : 0;
        }
    }
    int r[4], e[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) { r[k] = (int)(s0 + k) - d[k]; e[k] = d[k]; }
    while (e[0] | e[1] | e[2] | e[3]) {
#pragma unroll
        for (int k = 0; k < 4; ++k) e[k] = e[k] ? (int)__ldg(rel + r[k]) : 0;
#pragma unroll
        for (int k = 0; k < 4; ++k) r[k] -= e[k];
    }
#pragma unroll
    for (int k = 0; k < 4; ++k)
        if (d[k]) {
            const int lab = __ldg(idx_s + r[k]);
            labels[oi[k]] = lab;
            if (cnt) atomicAdd(cnt + lab, 1);
        }
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
                        const unsigned long long *dense_list, unsigned int *rel, const int *idx_s, Ctrl *ctrl,
                        int num_sms, const unsigned int *gate, cudaStream_t s)
{
    if (N <= 0) return cudaSuccess;
    const unsigned int grid = (unsigned int)min((int64_t)blocks_for(N, kLinkBlock), (int64_t)num_sms * FOF_LINK_MINB);
    // tickets sized so that every warp of the grid draws at least ~4 of them: with one or two per warp
    // (a few million particles) the slowest warp would carry twice the mean
    const int64_t per_warp = (N / 32) / (4 * (int64_t)grid * kWarpsPerCta);
    const unsigned int tile_batch = (unsigned int)min(max(per_warp / 2, (int64_t)1), (int64_t)kTileBatch);  // items are fewer and longer
    const unsigned int sparse_batch = (unsigned int)min(max(per_warp, (int64_t)1), (int64_t)kSparseBatch);
    link_kernel<<<grid, kLinkBlock, 0, s>>>(sorted, N, g, cell_start, dense_list, rel, idx_s, ctrl, tile_batch,
                                            sparse_batch, gate);
    return cudaGetLastError();
}

cudaError_t launch_write_labels(const unsigned int *rel, const int *idx_s, int *labels, int64_t N,
                                const unsigned int *gate, int *cnt, unsigned long long *state, int64_t state_items,
                                Ctrl *ctrl, cudaStream_t s)
{
    const bool vec = (((uintptr_t)rel | (uintptr_t)idx_s) & 15) == 0;
    if (N > 0)
        write_labels_kernel<<<blocks_for(N, kBlock * 4), kBlock, 0, s>>>(rel, idx_s, labels, N, vec, gate, cnt, state,
                                                                         state_items, ctrl);
    return cudaGetLastError();
}

}  // namespace fof
