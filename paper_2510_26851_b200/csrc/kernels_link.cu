// kernels_link.cu — H4 half-stencil pair tests + union, H5 flatten.
// What is linked: PAPER.md:85-87 (§2 step iv) and PAPER.md:200-214 (Alg. 2 candidate cells and
// mask); the 27-cell stencil with indices mod n is PAPER.md:202.  The T label sweeps of
// PAPER.md:221-225 are replaced by their fixed point, computed with a lock-free union-find on the
// label array (root = minimum original index = the converged min-label).
//
// Design: a CTA owns a tile of Sx x Sy x Sz home cells.  It stages the home cells
// and their half-stencil shell ((Sx+2) x (Sy+2) x (Sz+1) cells, each cell row one or two contiguous
// runs of the cell-sorted array) in shared memory, tests every (home particle, candidate) pair
// with W lanes per home particle walking the concatenated candidate ranges, and resolves the
// edges it finds in a shared-memory union-find.  Only the result leaves the CTA: one global
// union (particle, minimum original index of its local component) per staged particle that is in
// a non-trivial local component.  Tiles that do not fit the shared-memory capacity are flagged
// and handled by a per-particle global-memory kernel (same stencil, same predicate).
#include "fof_internal.cuh"

namespace fof {

// Half stencil: every unordered pair of distinct neighbouring cells is visited from exactly one
// side (needs n >= 3 so that +1 and -1 are different cells): the rows (dy, dz) = (-1,+1), (0,+1),
// (+1,+1), (+1,0) with dx in {-1,0,+1}, the +x neighbour in the home row, and the home cell
// itself (partners after me).
__constant__ int kRowDy[4] = {-1, 0, 1, 1};
__constant__ int kRowDz[4] = {1, 1, 1, 0};

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

// ---- shared-memory union-find over the staged particles (index = staged slot; root = smallest
// slot of the set).  Same lock-free scheme as the global one: CAS at roots, path halving.
__device__ __forceinline__ int find_s(volatile int *lab, int x)
{
    int p = lab[x];
    while (p != x) {
        const int gp = lab[p];
        if (gp != p) lab[x] = gp;
        x = p;
        p = gp;
    }
    return x;
}

__device__ __forceinline__ int unite_s(volatile int *lab, int a, int b)
{
    int ra = find_s(lab, a), rb = find_s(lab, b);
    while (ra != rb) {
        if (ra < rb) { const int t = ra; ra = rb; rb = t; }  // ra is the larger root
        const int old = atomicCAS(const_cast<int *>(lab) + ra, ra, rb);
        if (old == ra) return rb;
        ra = find_s(lab, old);
    }
    return ra;
}

// Full compression of both end points after a union (both are non-roots unless they are r).
__device__ __forceinline__ int unite_compress(volatile int *lab, int a, int b)
{
    const int r = unite_s(lab, a, b);
    if (a != r) lab[a] = r;
    if (b != r) lab[b] = r;
    return r;
}

// ---- mbarrier + bulk-copy (TMA 1-D) helpers: the staged rows are contiguous runs of float4 in
// the cell-sorted array, 16-byte aligned, so each run is ONE cp.async.bulk issued by one lane.
__device__ __forceinline__ unsigned int smem_u32(const void *p) { return (unsigned int)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long *mbar, unsigned int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(mbar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long *mbar, unsigned int bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(mbar)), "r"(bytes) : "memory");
}

__device__ __forceinline__ void bulk_copy_g2s(void *dst_smem, const void *src_gmem, unsigned int bytes,
                                              unsigned long long *mbar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(mbar))
                 : "memory");
}

__device__ __forceinline__ void mbar_wait(unsigned long long *mbar, unsigned int parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(mbar)),
        "r"(parity)
        : "memory");
}

constexpr int kMaxRows = 96;  // staged rows of a tile: (Sy+2)(Sz+1) <= 10 * 9

struct TileGeom {
    int x0, y0, z0;  // first home cell
    int sx, sy, sz;  // home cells of this tile (clipped at the grid edge)
    int W2, RY;      // staged cells per row, staged rows per z level
    int lxa, lxb;    // staged cells [lxa, lxb] of a row are one run of the sorted array (the main piece);
                     // lx < lxa is the cell n-1 reached through the periodic x face, lx > lxb is cell 0
};

// Staged-row descriptors (shared memory).  Slot of the first particle of staged cell lx of row r:
//   adj[r] + cell_start[cellbase[r] + lx]          for lxa <= lx <= lxb + 1
//   rowoff[r] / rowoff[r+1]                        for the wrapped end cells
struct RowTable {
    int cellbase[kMaxRows];
    int adj[kMaxRows];
    int rowoff[kMaxRows + 1];
};

template <bool WRAP>
__device__ __forceinline__ int slot_of(const unsigned int *__restrict__ cs, const RowTable &rt, int r, int lx,
                                       const TileGeom &tg)
{
    if (WRAP) {
        if (lx < tg.lxa) return rt.rowoff[r];
        if (lx > tg.lxb + 1) return rt.rowoff[r + 1];
    }
    return rt.adj[r] + (int)__ldg(cs + rt.cellbase[r] + lx);
}

// The five candidate ranges (staged slots) of one home particle: the rest of its own cell plus
// the +x cell, and the rows (dy,dz) = (-1,+1), (0,+1), (+1,+1), (+1,0) of three cells each --
// trimmed by the geometric reach filter: a neighbouring cell in direction (dx,dy,dz) can hold a
// partner only if the particle lies within `reach` (= b in cell units + slack) of the
// corresponding faces of its own cell.  A filtered-out cell cannot contain a pair with d2 <= b2,
// so the edge set is unchanged; a row stays one contiguous range because only its two end cells
// are trimmed.
struct Ranges {
    int beg[5], end[5];
    int K;  // candidates after the filter
};

// hr = staged row of the home cell, r1 = staged row (ly-1, lz+1); fx,fy,fz = position inside the
// home cell in cell units; lx = staged x index of the home cell.
template <bool WRAP>
__device__ __forceinline__ Ranges candidate_ranges(int si, int lx, float fx, float fy, float fz, int hr, int r1,
                                                   const unsigned int *__restrict__ cs, const RowTable &rt,
                                                   const TileGeom &tg, const Grid &g)
{
    Ranges R;
    const float lo = g.reach, hi = 1.0f - g.reach;
    const int xl = fx < lo, xh = fx > hi;  // can reach the cell at x-1 / x+1
    const bool yl = fy < lo, yh = fy > hi, zh = fz > hi;
    const int a = lx - xl, b = lx + 1 + xh;  // trimmed cell span [a, b) of a neighbour row
    R.beg[0] = si + 1;
    R.end[0] = slot_of<WRAP>(cs, rt, hr, b, tg);
    R.beg[1] = R.end[1] = R.beg[2] = R.end[2] = R.beg[3] = R.end[3] = R.beg[4] = R.end[4] = 0;
    if (zh) {
        if (yl) { R.beg[1] = slot_of<WRAP>(cs, rt, r1, a, tg); R.end[1] = slot_of<WRAP>(cs, rt, r1, b, tg); }
        R.beg[2] = slot_of<WRAP>(cs, rt, r1 + 1, a, tg); R.end[2] = slot_of<WRAP>(cs, rt, r1 + 1, b, tg);
        if (yh) { R.beg[3] = slot_of<WRAP>(cs, rt, r1 + 2, a, tg); R.end[3] = slot_of<WRAP>(cs, rt, r1 + 2, b, tg); }
    }
    if (yh) { R.beg[4] = slot_of<WRAP>(cs, rt, hr + 1, a, tg); R.end[4] = slot_of<WRAP>(cs, rt, hr + 1, b, tg); }
    R.K = (R.end[0] - R.beg[0]) + (R.end[1] - R.beg[1]) + (R.end[2] - R.beg[2]) + (R.end[3] - R.beg[3]) +
          (R.end[4] - R.beg[4]);
    return R;
}

constexpr int kLightMax = 8;  // home particles with at most this many candidates are tested by one thread

// Pass A: one warp per home row (rows handed out dynamically), one lane per home particle.  Light
// particles are finished here; the others are queued for pass B: the first particle of a cell
// ("leader") at the front of s_heavy, the rest at its back.
template <bool WRAP>
__device__ __forceinline__ void tile_pass_a(const float4 *s_pos, volatile int *s_lab, unsigned short *s_heavy,
                                            int cap, int *s_cnt, const unsigned int *__restrict__ cs,
                                            const RowTable &rt, const TileGeom &tg, const Grid &g,
                                            unsigned int &edges, unsigned int &ntests)
{
    const int lane = threadIdx.x & 31;
    const int R = tg.sy * tg.sz;
    const float inv_sy = 1.0f / (float)tg.sy;
    while (true) {
        int r = 0;
        if (lane == 0) r = atomicAdd(s_cnt + 0, 1);
        r = __shfl_sync(0xffffffffu, r, 0);
        if (r >= R) break;
        const int lz = (int)(((float)r + 0.5f) * inv_sy), ly = 1 + r - lz * tg.sy;
        const int hr = lz * tg.RY + ly, r1 = (lz + 1) * tg.RY + ly - 1;
        const float cyf = (float)(tg.y0 + ly - 1), czf = (float)(tg.z0 + lz);
        const int hbeg = slot_of<WRAP>(cs, rt, hr, 1, tg);
        const int cnt = slot_of<WRAP>(cs, rt, hr, tg.sx + 1, tg) - hbeg;
        for (int q = lane; q < cnt; q += 32) {
            const int si = hbeg + q;
            const float4 me = s_pos[si];
            const float ux = __fmul_rn(me.x, g.inv_cell);
            const int cx = min(__float2int_rd(ux), g.n_minus_1);
            const int lx = cx - tg.x0 + 1;
            const Ranges rg = candidate_ranges<WRAP>(si, lx, ux - (float)cx, fmaf(me.y, g.inv_cell, -cyf),
                                                     fmaf(me.z, g.inv_cell, -czf), hr, r1, cs, rt, tg, g);
            if (rg.K == 0) continue;
            if (rg.K > kLightMax) {
                const bool leader = si == slot_of<WRAP>(cs, rt, hr, lx, tg);
                if (leader) s_heavy[atomicAdd(s_cnt + 1, 1)] = (unsigned short)si;
                else s_heavy[cap - 1 - atomicAdd(s_cnt + 2, 1)] = (unsigned short)si;
                continue;
            }
            ntests += (unsigned int)rg.K;
            int myroot = s_lab[si];
#pragma unroll
            for (int k = 0; k < 5; ++k) {
                for (int t = rg.beg[k]; t < rg.end[k]; ++t) {
                    const float4 pj = s_pos[t];
                    if (linked_t<WRAP>(me, pj, g)) {
                        ++edges;
                        if (s_lab[t] != myroot) myroot = unite_compress(s_lab, si, t);
                    }
                }
            }
        }
    }
}

// Pass B: queued home particles s_heavy[first + q * dir], q < count; W lanes each, walking the
// concatenated ranges with stride W.
template <int W, bool WRAP>
__device__ __forceinline__ void tile_pass_b(const float4 *s_pos, volatile int *s_lab, const unsigned short *s_heavy,
                                            int first, int dir, int count, int *s_next,
                                            const unsigned int *__restrict__ cs, const RowTable &rt,
                                            const TileGeom &tg, const Grid &g, unsigned int &edges,
                                            unsigned int &ntests)
{
    constexpr int G = 32 / W;
    const int lane = threadIdx.x & 31;
    const int grp = lane / W, gl = lane % W;
    while (true) {
        int q0 = 0;
        if (lane == 0) q0 = atomicAdd(s_next, G);
        q0 = __shfl_sync(0xffffffffu, q0, 0);
        if (q0 >= count) break;
        const int q = q0 + grp;
        if (q < count) {
            const int si = s_heavy[first + q * dir];
            const float4 me = s_pos[si];
            const float ux = __fmul_rn(me.x, g.inv_cell), uy = __fmul_rn(me.y, g.inv_cell),
                        uz = __fmul_rn(me.z, g.inv_cell);
            const int cx = min(__float2int_rd(ux), g.n_minus_1), cy = min(__float2int_rd(uy), g.n_minus_1),
                      cz = min(__float2int_rd(uz), g.n_minus_1);
            const int lx = cx - tg.x0 + 1, ly = cy - tg.y0 + 1, lz = cz - tg.z0;
            const Ranges rg = candidate_ranges<WRAP>(si, lx, ux - (float)cx, uy - (float)cy, uz - (float)cz,
                                                     lz * tg.RY + ly, (lz + 1) * tg.RY + ly - 1, cs, rt, tg, g);
            if (gl == 0) ntests += (unsigned int)rg.K;
            int myroot = s_lab[si];
            int off = gl;
#pragma unroll
            for (int k = 0; k < 5; ++k) {
                int t = rg.beg[k] + off;
                for (; t < rg.end[k]; t += W) {
                    const float4 pj = s_pos[t];
                    if (linked_t<WRAP>(me, pj, g)) {
                        ++edges;
                        if (s_lab[t] != myroot) myroot = unite_compress(s_lab, si, t);
                    }
                }
                off = t - rg.end[k];
            }
        }
    }
}

// flatten the shared-memory forest: s_lab[p] <- root(p).  Read-only walk (a halving store racing
// with the flatten store could leave a non-root behind).
__device__ __forceinline__ void tile_flatten(volatile int *s_lab, int total)
{
    for (int p = threadIdx.x; p < total; p += kLinkBlock) {
        int r = p, q;
        while ((q = s_lab[r]) != r) r = q;
        if (r != p) s_lab[p] = r;
    }
}

template <int W, bool WRAP>
__device__ __forceinline__ void tile_link(const float4 *s_pos, volatile int *s_lab, unsigned short *s_heavy, int cap,
                                          int total, int *s_cnt, const unsigned int *__restrict__ cs,
                                          const RowTable &rt, const TileGeom &tg, const Grid &g,
                                          unsigned int &edges, unsigned int &ntests)
{
    tile_pass_a<WRAP>(s_pos, s_lab, s_heavy, cap, s_cnt, cs, rt, tg, g, edges, ntests);
    __syncthreads();
    const int nlead = s_cnt[1], nrest = s_cnt[2];
    if (nlead) {
        // the leaders first: they hook most of their (dense) cells under themselves ...
        tile_pass_b<W, WRAP>(s_pos, s_lab, s_heavy, 0, 1, nlead, s_cnt + 3, cs, rt, tg, g, edges, ntests);
        __syncthreads();
        // ... so that after a flatten the remaining heavy particles mostly see lab[t] == lab[si]
        tile_flatten(s_lab, total);
        __syncthreads();
    }
    if (nrest) tile_pass_b<W, WRAP>(s_pos, s_lab, s_heavy, cap - 1, -1, nrest, s_cnt + 4, cs, rt, tg, g, edges, ntests);
}

template <int W>
__global__ void __launch_bounds__(kLinkBlock, 3) link_tile_kernel(const float4 *__restrict__ sorted, Grid g, Tile tp,
                                                                  const unsigned int *__restrict__ cell_start,
                                                                  int *parent, unsigned char *tile_flags, Ctrl *ctrl)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4 *s_pos = reinterpret_cast<float4 *>(smem_raw);
    int *s_labi = reinterpret_cast<int *>(s_pos + tp.cap);
    unsigned short *s_heavy = reinterpret_cast<unsigned short *>(s_labi + tp.cap);  // [cap]
    volatile int *s_lab = s_labi;
    __shared__ RowTable rt;
    __shared__ __align__(8) unsigned long long s_mbar;
    __shared__ int s_cnt[8];  // 0: next home row, 1: leaders, 2: other heavy, 3/4: pass-B tickets, 5: overflow
    __shared__ unsigned int s_edges, s_tests;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n = g.n;
    TileGeom tg;
    {
        const int t = blockIdx.x;
        const int tix = t % tp.tx, tiy = (t / tp.tx) % tp.ty, tiz = t / (tp.tx * tp.ty);
        tg.x0 = tix * tp.Sx; tg.y0 = tiy * tp.Sy; tg.z0 = tiz * tp.Sz;
        tg.sx = min(tp.Sx, n - tg.x0); tg.sy = min(tp.Sy, n - tg.y0); tg.sz = min(tp.Sz, n - tg.z0);
        tg.W2 = tg.sx + 2; tg.RY = tg.sy + 2;
        tg.lxa = tg.x0 == 0 ? 1 : 0;
        tg.lxb = tg.x0 + tg.sx == n ? tg.W2 - 2 : tg.W2 - 1;
    }
    const int nrows = tg.RY * (tg.sz + 1);
    if (tid == 0) {
        mbar_init(&s_mbar, 1);
        s_edges = 0; s_tests = 0;
    }
    if (tid < 8) s_cnt[tid] = 0;
    __syncthreads();

    // ---- 1. row table + staging, by warp 0: every staged row is up to three runs of the sorted
    // array (cell n-1 through the periodic x face | main piece | cell 0); the copies are bulk
    // asynchronous copies that land on s_mbar.  Row (ly=0, lz=0) is not in the half stencil.
    if (warp == 0) {
        unsigned int gb[3][3], len[3][3];  // [row slot of this lane][piece]
        int carry = 0;
#pragma unroll
        for (int it = 0; it < 3; ++it) {
            const int r = it * 32 + lane;
            int cnt = 0;
            len[it][0] = len[it][1] = len[it][2] = 0;
            gb[it][0] = gb[it][1] = gb[it][2] = 0;
            int cellbase = 0;
            if (r < nrows) {
                const int lz = r / tg.RY, ly = r - lz * tg.RY;
                int gy = tg.y0 - 1 + ly; gy = gy < 0 ? gy + n : (gy >= n ? gy - n : gy);
                int gz = tg.z0 + lz; gz = gz >= n ? gz - n : gz;
                const int rowbase = n * (gy + n * gz);
                cellbase = rowbase + tg.x0 - 1;
                if (!(ly == 0 && lz == 0)) {
                    gb[it][1] = __ldg(cell_start + cellbase + tg.lxa);
                    len[it][1] = __ldg(cell_start + cellbase + tg.lxb + 1) - gb[it][1];
                    if (tg.lxa) {
                        gb[it][0] = __ldg(cell_start + rowbase + n - 1);
                        len[it][0] = __ldg(cell_start + rowbase + n) - gb[it][0];
                    }
                    if (tg.lxb == tg.W2 - 2) {
                        gb[it][2] = __ldg(cell_start + rowbase);
                        len[it][2] = __ldg(cell_start + rowbase + 1) - gb[it][2];
                    }
                    cnt = (int)(len[it][0] + len[it][1] + len[it][2]);
                }
            }
            int incl = cnt;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int v = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += v;
            }
            const int off = carry + incl - cnt;
            if (r < nrows) {
                rt.rowoff[r] = off;
                rt.cellbase[r] = cellbase;
                rt.adj[r] = off + (int)len[it][0] - (int)gb[it][1];
            }
            gb[it][0] = (unsigned int)off;  // reuse: staged slot of the row (piece 0 source index is re-read below)
            carry += __shfl_sync(0xffffffffu, incl, 31);
            if (it * 32 + 32 >= nrows) break;
        }
        const int total = carry;
        if (lane == 0) {
            rt.rowoff[nrows] = total;
            if (total > tp.cap) {  // does not fit: leave this tile to link_overflow_kernel
                s_cnt[5] = 1;
                tile_flags[blockIdx.x] = 1;
                atomicAdd(&ctrl->overflow_tiles, 1u);
            } else if (total > 0) {
                mbar_arrive_expect_tx(&s_mbar, (unsigned int)total * 16u);
            }
        }
        __syncwarp();
        if (total > 0 && total <= tp.cap) {
#pragma unroll
            for (int it = 0; it < 3; ++it) {
                const int r = it * 32 + lane;
                if (r < nrows) {
                    int dst = (int)gb[it][0];
                    if (len[it][0]) {
                        const int lz = r / tg.RY, ly = r - lz * tg.RY;
                        int gy = tg.y0 - 1 + ly; gy = gy < 0 ? gy + n : (gy >= n ? gy - n : gy);
                        int gz = tg.z0 + lz; gz = gz >= n ? gz - n : gz;
                        const unsigned int src = __ldg(cell_start + n * (gy + n * gz) + n - 1);
                        bulk_copy_g2s(s_pos + dst, sorted + src, len[it][0] * 16u, &s_mbar);
                        dst += (int)len[it][0];
                    }
                    if (len[it][1]) {
                        bulk_copy_g2s(s_pos + dst, sorted + gb[it][1], len[it][1] * 16u, &s_mbar);
                        dst += (int)len[it][1];
                    }
                    if (len[it][2]) bulk_copy_g2s(s_pos + dst, sorted + gb[it][2], len[it][2] * 16u, &s_mbar);
                }
                if (it * 32 + 32 >= nrows) break;
            }
        }
    }
    __syncthreads();
    const int total = rt.rowoff[nrows];
    if (total == 0 || s_cnt[5]) return;
    for (int p = tid; p < total; p += kLinkBlock) s_labi[p] = p;
    mbar_wait(&s_mbar, 0);
    __syncthreads();

    // ---- 2. pair tests + shared-memory unions
    unsigned int edges = 0, ntests = 0;
    const bool wrap_tile = (n < 6) || tg.x0 < 1 || tg.x0 + tg.sx > n - 1 || tg.y0 < 1 || tg.y0 + tg.sy > n - 1 ||
                           tg.z0 + tg.sz > n - 1;
    if (wrap_tile) tile_link<W, true>(s_pos, s_lab, s_heavy, tp.cap, total, s_cnt, cell_start, rt, tg, g, edges, ntests);
    else tile_link<W, false>(s_pos, s_lab, s_heavy, tp.cap, total, s_cnt, cell_start, rt, tg, g, edges, ntests);
    __syncthreads();

    // ---- 3. hand the local components to the global union-find (parent[] on original indices):
    // flatten; roots park their own original index in s_lab as ~idx; every member lowers the w slot of
    // its root to the minimum original index m of the component; unite(idx, m) for everyone.
    tile_flatten(s_lab, total);
    __syncthreads();
    for (int p = tid; p < total; p += kLinkBlock)
        if (s_lab[p] == p) s_lab[p] = ~__float_as_int(s_pos[p].w);
    __syncthreads();
    int *s_w = reinterpret_cast<int *>(s_pos);
    for (int p = tid; p < total; p += kLinkBlock) {
        const int l = s_lab[p];
        if (l >= 0) atomicMin(s_w + 4 * l + 3, s_w[4 * p + 3]);
    }
    __syncthreads();
    for (int p = tid; p < total; p += kLinkBlock) {
        const int l = s_lab[p];
        int a, m;
        if (l >= 0) { a = s_w[4 * p + 3]; m = s_w[4 * l + 3]; }
        else { a = ~l; m = s_w[4 * p + 3]; }
        if (a != m) unite(parent, a, m);
    }

    // ---- counters: one set of global atomics per CTA
    for (int o = 16; o > 0; o >>= 1) {
        edges += __shfl_xor_sync(0xffffffffu, edges, o);
        ntests += __shfl_xor_sync(0xffffffffu, ntests, o);
    }
    if (lane == 0) { atomicAdd(&s_edges, edges); atomicAdd(&s_tests, ntests); }
    __syncthreads();
    if (tid == 0) {
        if (s_edges) atomicAdd(&ctrl->edges, (unsigned long long)s_edges);
        if (s_tests) atomicAdd(&ctrl->pair_tests, (unsigned long long)s_tests);
    }
}

// ---------------------------------------------------------------------------------------------
// Overflow path: one thread per cell-sorted particle of a flagged tile, candidates read from
// global memory, every edge united directly in the global union-find.
// ---------------------------------------------------------------------------------------------
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

__global__ void __launch_bounds__(kLinkBlock) link_overflow_kernel(const float4 *__restrict__ sorted, int64_t N,
                                                                   Grid g, Tile tp,
                                                                   const unsigned int *__restrict__ cell_start,
                                                                   int *parent,
                                                                   const unsigned char *__restrict__ tile_flags,
                                                                   Ctrl *ctrl)
{
    if (ctrl->overflow_tiles == 0) return;
    PairCounters pc = {0u, 0u};
    const int n = g.n;
    for (int64_t s = (int64_t)blockIdx.x * kLinkBlock + threadIdx.x; s < N; s += (int64_t)gridDim.x * kLinkBlock) {
        const float4 me = __ldg(sorted + s);
        const int cx = cell1(me.x, g), cy = cell1(me.y, g), cz = cell1(me.z, g);
        const int tile = cx / tp.Sx + tp.tx * (cy / tp.Sy + tp.ty * (cz / tp.Sz));
        if (!tile_flags[tile]) continue;
        const int oi = __float_as_int(me.w);
        const int xm = cx == 0 ? n - 1 : cx - 1, xp = cx == n - 1 ? 0 : cx + 1;
        const unsigned int home = cell_id(cx, cy, cz, n);
        test_range(sorted, (unsigned int)s + 1, __ldg(cell_start + home + 1), me, oi, g, parent, pc);
        {
            const unsigned int c = cell_id(xp, cy, cz, n);
            test_range(sorted, __ldg(cell_start + c), __ldg(cell_start + c + 1), me, oi, g, parent, pc);
        }
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            int ny = cy + kRowDy[r], nz = cz + kRowDz[r];
            ny = ny < 0 ? n - 1 : (ny >= n ? 0 : ny);
            nz = nz >= n ? 0 : nz;
            const int xs[3] = {xm, cx, xp};
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const unsigned int c = cell_id(xs[k], ny, nz, n);
                test_range(sorted, __ldg(cell_start + c), __ldg(cell_start + c + 1), me, oi, g, parent, pc);
            }
        }
    }
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

// P_exec of DESIGN.md §7: candidate pairs the unfiltered half stencil implies on this grid,
// sum over cells of occ (occ - 1) / 2 + occ * (occupancy of the 13 half-stencil cells).  Run by
// fof_link_stats only (not on the hot path).
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

template <int W>
static cudaError_t launch_tiles(const float4 *sorted, Grid g, Tile tp, size_t smem, int64_t ntiles,
                                const unsigned int *cell_start, int *labels, unsigned char *tile_flags, Ctrl *ctrl,
                                cudaStream_t s)
{
    static size_t configured = 0;  // largest dynamic shared memory size this instantiation was opted in for
    if (smem > configured) {
        cudaError_t e = cudaFuncSetAttribute(link_tile_kernel<W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured = smem;
    }
    link_tile_kernel<W><<<(unsigned int)ntiles, kLinkBlock, smem, s>>>(sorted, g, tp, cell_start, labels, tile_flags,
                                                                      ctrl);
    return cudaGetLastError();
}

cudaError_t launch_link(const float4 *sorted, int64_t N, Grid g, Tile tp, size_t smem, int w, int64_t ntiles,
                        const unsigned int *cell_start, int *labels, unsigned char *tile_flags, Ctrl *ctrl,
                        int num_sms, cudaStream_t s)
{
    if (N <= 0) return cudaSuccess;
    cudaError_t e;
    switch (w) {
    case 4: e = launch_tiles<4>(sorted, g, tp, smem, ntiles, cell_start, labels, tile_flags, ctrl, s); break;
    case 16: e = launch_tiles<16>(sorted, g, tp, smem, ntiles, cell_start, labels, tile_flags, ctrl, s); break;
    case 32: e = launch_tiles<32>(sorted, g, tp, smem, ntiles, cell_start, labels, tile_flags, ctrl, s); break;
    default: e = launch_tiles<8>(sorted, g, tp, smem, ntiles, cell_start, labels, tile_flags, ctrl, s); break;
    }
    if (e != cudaSuccess) return e;
    const unsigned int grid = (unsigned int)min((int64_t)blocks_for(N, kLinkBlock), (int64_t)num_sms * 8);
    link_overflow_kernel<<<grid, kLinkBlock, 0, s>>>(sorted, N, g, tp, cell_start, labels, tile_flags, ctrl);
    return cudaGetLastError();
}

cudaError_t launch_flatten(int *labels, int64_t N, cudaStream_t s)
{
    if (N > 0) flatten_kernel<<<blocks_for(N, kBlock), kBlock, 0, s>>>(labels, N);
    return cudaGetLastError();
}

}  // namespace fof
