// kernels_block.cu — the BLOCK PATH of H1-H5: one partition pass into spatial blocks, then one CTA per block
// that cell-sorts and links its particles entirely in shared memory.
// What is computed is unchanged: PAPER.md:193-199 (wrap, grid, cell index, sort by cell)
// (candidate cells of the 27 stencil, minimum-image mask d^2 <= b^2), PAPER.md:221-225 (label sweeps, here
// their fixed point by union-find), PAPER.md:91 / 180 (label = minimum original index).
//
// Why: measured on B200, a scattered 16-byte store costs the same ~12 ps chip-wide whatever
// the number of open streams (80 G records/s), so the two scatter passes of the cell path (bin-contiguous, then
// cell-contiguous) cost ~0.5 ms at 256^3 however they are tuned, and the link kernel then gathers candidates
// from global memory.  Here every record is scattered ONCE, to its block (2^sx x 2^sy x 2^sz cells, a few
// thousand particles), and a particle within `reach` of a backward face of its block is ALSO written, as a ghost,
// to the block(s) behind that face.  A block then owns every pair (own, own) and (own, ghost): each unordered
// pair of particles in adjacent cells is tested by exactly one block (the backward one), and nothing that a CTA
// needs lives outside its contiguous slice of the record array, which TMA brings in with one bulk copy.
//   block_scatter_kernel  records to their blocks (fixed slices, shared cursors)   pos -> part, labels[i] = i;
//                         sets ctrl->mode = 1 if a block overflows its slice (the cell path then runs)
//   block_link_kernel     TMA load, counting sort by local cell in shared memory, half-stencil tests,
//                         union-find in shared memory rooted at the minimum ORIGINAL index; writes
//                         labels[own non-root] = original index of its local root, lists one equivalence
//                         (ghost, local root) per linked ghost
//   cross_link_kernel     unions of the listed equivalences on `labels` (global lock-free union-find)
//   flatten_labels_kernel labels[i] = root(i)
#include "fof_internal.cuh"

namespace fof {

namespace {

constexpr unsigned int kFull = 0xffffffffu;
#ifdef FOF_BLOCK_TIMING
__device__ unsigned long long g_dbg[16];
#define DBG_T(var) const long long var = clock64()
#define DBG_ADD(k, a, b) do { if ((threadIdx.x & 31u) == 0) atomicAdd(&g_dbg[k], (unsigned long long)((b) - (a))); } while (0)
#else
#define DBG_T(var)
#define DBG_ADD(k, a, b)
#endif

// ---- which blocks get a copy of a particle ---------------------------------------------------------------
// H = forward half of the 26 block offsets: (1,0,0), (*,1,0), (*,*,1).  Block A tests (own of A) x (own of
// A + d) for d in H, so a particle of block P is exported to P - d, i.e. in the directions e in -H:
// (-1,0,0), (*,-1,0), (*,*,-1), and only if it lies within `reach` of every face it has to cross.
template <typename F>
__device__ __forceinline__ unsigned int classify(float x, float y, float z, const Grid &g, const BlockGeom &bg, F ghost)
{
    const float ux = __fmul_rn(x, g.inv_cell), uy = __fmul_rn(y, g.inv_cell), uz = __fmul_rn(z, g.inv_cell);
    const int cx = min(max(__float2int_rd(ux), 0), g.n_minus_1);
    const int cy = min(max(__float2int_rd(uy), 0), g.n_minus_1);
    const int cz = min(max(__float2int_rd(uz), 0), g.n_minus_1);
    const int bx = cx >> bg.sx, by = cy >> bg.sy, bz = cz >> bg.sz;
    const float lo = g.reach;
    const int mx = (1 << bg.sx) - 1, my = (1 << bg.sy) - 1, mz = (1 << bg.sz) - 1;
    const bool xl = ((cx & mx) == 0) & (ux - (float)cx < lo);
    const bool yl = ((cy & my) == 0) & (uy - (float)cy < lo);
    const bool zl = ((cz & mz) == 0) & (uz - (float)cz < lo);
    if (xl | yl | zl) {
        const float hi = 1.0f - g.reach;
        const bool xh = (((cx & mx) == mx) | (cx == g.n_minus_1)) & (ux - (float)cx > hi);
        const bool yh = (((cy & my) == my) | (cy == g.n_minus_1)) & (uy - (float)cy > hi);
        for (int ez = 0; ez >= -1; --ez) {
            if (ez && !zl) continue;
            for (int ey = -1; ey <= 1; ++ey) {
                if (ey && !(ey < 0 ? yl : yh)) continue;
                for (int ex = -1; ex <= 1; ++ex) {
                    if (ex && !(ex < 0 ? xl : xh)) continue;
                    if (ez == 0 && !(ey == -1 || (ey == 0 && ex == -1))) continue;  // e must be in -H
                    int qx = bx + ex, qy = by + ey, qz = bz + ez;
                    qx = qx < 0 ? bg.nbx - 1 : (qx >= bg.nbx ? 0 : qx);
                    qy = qy < 0 ? bg.nby - 1 : (qy >= bg.nby ? 0 : qy);
                    qz = qz < 0 ? bg.nbz - 1 : qz;
                    ghost((unsigned int)(qx + bg.nbx * (qy + bg.nby * qz)));
                }
            }
        }
    }
    return (unsigned int)(bx + bg.nbx * (by + bg.nby * bz));
}

__device__ __forceinline__ void wrap3(float &x, float &y, float &z, const Grid &g, bool &bad)
{
    if (!(isfinite(x) && isfinite(y) && isfinite(z))) { bad = true; x = y = z = 0.0f; }
    x = wrap1(x, g.L);
    y = wrap1(y, g.L);
    z = wrap1(z, g.L);
}

// ---------------------------------------------------------------------------------------------------------
// records to their blocks.  Block b owns the fixed slice part[b cap, (b + 1) cap) (no histogram pass, no offsets:
// the plan sizes the blocks so that a block holds about half of what fits; a block that overflows sets
// ctrl->mode = 1 and the cell path runs instead).  A CTA takes tiles of TH x PER particles (registers); the rank
// of a record among the tile's records of its block comes from a shared-memory counter, the tile's slots from
// ONE global atomic per (tile, block) on the block's cursor, issued by the thread that drew rank 0: all CTAs
// append to the same few thousand open lines, which the L2 merges before they reach DRAM (measured, 2^24 records
// into 4096 blocks: private per-CTA streams 0.42 ms, shared cursors 0.25 ms; a scattered 16-byte store costs the
// same ~12 ps chip-wide whatever the pattern).  Only the counters a tile touched are read and cleared again, so
// the cost of a tile does not depend on the number of blocks.  The rare ghost copies take one global atomic each.
// ---------------------------------------------------------------------------------------------------------
#ifndef FOF_SCAT_THREADS
#define FOF_SCAT_THREADS 512
#endif
#ifndef FOF_SCAT_PER
#define FOF_SCAT_PER 4
#endif
#ifndef FOF_SCAT_MINB
#define FOF_SCAT_MINB 3
#endif
#ifndef FOF_SCAT_CTAS
#define FOF_SCAT_CTAS 3
#endif
constexpr int kScatThreads = FOF_SCAT_THREADS, kScatPer = FOF_SCAT_PER;

template <bool VEC>
__global__ void __launch_bounds__(kScatThreads, FOF_SCAT_MINB) block_scatter_kernel(const float *__restrict__ pos, int64_t N, Grid g,
                                                                     BlockGeom bg, unsigned int *cursor,
                                                                     float4 *__restrict__ part, unsigned int cap,
                                                                     int *__restrict__ labels, bool labels_vec,
                                                                     int *__restrict__ cnt, Ctrl *ctrl)
{
    extern __shared__ unsigned int s_cnt[];  // [bins]: records of the current tile per block, then the tile's first slot
    __shared__ unsigned int s_tile;
    constexpr int T = kScatThreads * kScatPer;
    const int64_t ntiles = (N + T - 1) / T;
    const int tid = threadIdx.x;
    for (int b = tid; b < bg.bins; b += kScatThreads) s_cnt[b] = 0u;
    bool bad = false, over = false;
    for (;;) {
        __syncthreads();
        if (tid == 0) s_tile = atomicAdd(&ctrl->tile_ticket2, 1u);
        __syncthreads();
        const int64_t tile = s_tile;
        if (tile >= ntiles) break;
        const int64_t base = tile * T;
        float4 rec[kScatPer];
        unsigned int bin[kScatPer], rank[kScatPer];
#pragma unroll
        for (int q = 0; q < kScatPer / 4; ++q) {
            const int64_t i = base + ((int64_t)q * kScatThreads + tid) * 4;
            if (VEC && i + 4 <= N) {
                const float4 *p = reinterpret_cast<const float4 *>(pos + 3 * i);
                const float4 a = __ldg(p), b = __ldg(p + 1), c = __ldg(p + 2);
                rec[4 * q] = make_float4(a.x, a.y, a.z, __int_as_float((int)i));
                rec[4 * q + 1] = make_float4(a.w, b.x, b.y, __int_as_float((int)i + 1));
                rec[4 * q + 2] = make_float4(b.z, b.w, c.x, __int_as_float((int)i + 2));
                rec[4 * q + 3] = make_float4(c.y, c.z, c.w, __int_as_float((int)i + 3));
            } else {
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const int64_t j = i + k;
                    rec[4 * q + k] = j < N ? make_float4(__ldg(pos + 3 * j), __ldg(pos + 3 * j + 1), __ldg(pos + 3 * j + 2),
                                                         __int_as_float((int)j))
                                           : make_float4(0.f, 0.f, 0.f, __int_as_float(-1));
                }
            }
            // H5, first half: labels[i] = i (final for every singleton), coalesced; the size counters of H6 start at 0
            if (labels_vec && i + 4 <= N) *reinterpret_cast<int4 *>(labels + i) = make_int4((int)i, (int)i + 1, (int)i + 2, (int)i + 3);
            else
                for (int k = 0; k < 4; ++k) if (i + k < N) labels[i + k] = (int)(i + k);
            if (i + 4 <= N) *reinterpret_cast<int4 *>(cnt + i) = make_int4(0, 0, 0, 0);  // workspace array: aligned
            else
                for (int k = 0; k < 4; ++k) if (i + k < N) cnt[i + k] = 0;
        }
#pragma unroll
        for (int k = 0; k < kScatPer; ++k) {
            bin[k] = 0xffffffffu;
            if (__float_as_int(rec[k].w) >= 0) {
                wrap3(rec[k].x, rec[k].y, rec[k].z, g, bad);
                const float4 r = rec[k];
                bin[k] = classify(r.x, r.y, r.z, g, bg, [&](unsigned int gb) {
                    const unsigned int at = atomicAdd(&cursor[gb], 1u);
                    if (at < cap) part[(size_t)gb * cap + at] = make_float4(r.x, r.y, r.z, __uint_as_float(__float_as_uint(r.w) | kGhostBit));
                    else over = true;
                });
                rank[k] = atomicAdd(&s_cnt[bin[k]], 1u);
            }
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < kScatPer; ++k)
            if (bin[k] != 0xffffffffu && rank[k] == 0u) {  // I drew the first rank: I fetch the tile's slots of this block
                const unsigned int c = s_cnt[bin[k]];
                const unsigned int at = atomicAdd(&cursor[bin[k]], c);
                if (at + c > cap) over = true;
                s_cnt[bin[k]] = at;
            }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < kScatPer; ++k)
            if (bin[k] != 0xffffffffu) {
                const unsigned int at = s_cnt[bin[k]] + rank[k];
                if (at < cap) part[(size_t)bin[k] * cap + at] = rec[k];
            }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < kScatPer; ++k)
            if (bin[k] != 0xffffffffu && rank[k] == 0u) s_cnt[bin[k]] = 0u;
    }
    if (bad) atomicOr(&ctrl->error, 1u);
    if (over) ctrl->mode = 1u;
}

// ---------------------------------------------------------------------------------------------------------
// block_link_kernel
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned int smem_u32(const void *p) { return (unsigned int)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned int bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned int parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// TMA bulk copy global -> shared (contiguous, 16-byte granular), completion on an mbarrier
__device__ __forceinline__ void tma_load_1d(void *dst, const void *src, unsigned int bytes, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// union-find over the block's slots in shared memory; the root of a set is its member with the smallest
// ORIGINAL index (w with the ghost bit masked), so a parent always has the smaller original index: hooks are
// atomicCAS on roots, halving stores are benign (same argument as find_rel / unite_rel in fof_internal.cuh).
__device__ __forceinline__ int find_s(volatile unsigned int *par, int x)
{
    int p = (int)par[x];
    while (p != x) {
        const int gp = (int)par[p];
        if (gp != p) par[x] = (unsigned int)gp;
        x = p;
        p = gp;
    }
    return x;
}
__device__ __forceinline__ unsigned int orig_of(const float4 *rec, int s) { return __float_as_uint(rec[s].w) & ~kGhostBit; }

__device__ __forceinline__ int unite_s(unsigned int *par, const float4 *rec, int a, int b)
{
    int ra = find_s(par, a), rb = find_s(par, b);
    while (ra != rb) {
        if (orig_of(rec, ra) < orig_of(rec, rb)) { const int t = ra; ra = rb; rb = t; }  // ra: larger original index
        const unsigned int old = atomicCAS(par + ra, (unsigned int)ra, (unsigned int)rb);
        if (old == (unsigned int)ra) { ra = rb; break; }
        ra = find_s(par, (int)old);
    }
    // both ends straight under the root (an ancestor with a smaller original index: still a forest), so that
    // the next test of par[j] against the cached root succeeds
    if (a != ra) ((volatile unsigned int *)par)[a] = (unsigned int)ra;
    if (b != ra) ((volatile unsigned int *)par)[b] = (unsigned int)ra;
    return ra;
}

template <bool WRAP>
__device__ __forceinline__ bool linked_b(const float4 &a, const float4 &b, const Grid &g)
{
    float dx = __fsub_rn(a.x, b.x), dy = __fsub_rn(a.y, b.y), dz = __fsub_rn(a.z, b.z);
    if (WRAP) {  // the selects of min_image, branch-free (same values: one shift by -+L where |d| > L/2)
        const float nh = -g.h;
        dx = dx > g.h ? __fsub_rn(dx, g.L) : (dx < nh ? __fadd_rn(dx, g.L) : dx);
        dy = dy > g.h ? __fsub_rn(dy, g.L) : (dy < nh ? __fadd_rn(dy, g.L) : dy);
        dz = dz > g.h ? __fsub_rn(dz, g.L) : (dz < nh ? __fadd_rn(dz, g.L) : dz);
    }
    const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
    return d2 <= g.b2;
}

struct BlockOrigin { int x0, y0, z0, ncx, ncy, ncz; };  // first own cell and number of own cells per axis

// local cell (lx, ly, lz) of a record of this block: own cells are lx in [1, ncx], ly in [1, ncy], lz in
// [0, ncz); ghosts sit in the layers lx = 0 / ncx + 1, ly = 0 / ncy + 1, lz = ncz (periodic images folded)
__device__ __forceinline__ void local_cell(const float4 &r, const Grid &g, const BlockGeom &bg, const BlockOrigin &o,
                                           int &lx, int &ly, int &lz, float &fx, float &fy, float &fz)
{
    const float ux = __fmul_rn(r.x, g.inv_cell), uy = __fmul_rn(r.y, g.inv_cell), uz = __fmul_rn(r.z, g.inv_cell);
    const int cx = min(max(__float2int_rd(ux), 0), g.n_minus_1);
    const int cy = min(max(__float2int_rd(uy), 0), g.n_minus_1);
    const int cz = min(max(__float2int_rd(uz), 0), g.n_minus_1);
    fx = ux - (float)cx; fy = uy - (float)cy; fz = uz - (float)cz;
    lx = cx - o.x0 + 1; ly = cy - o.y0 + 1; lz = cz - o.z0;
    if (lx < 0) lx += g.n; else if (lx >= bg.X) lx -= g.n;
    if (ly < 0) ly += g.n; else if (ly >= bg.Y) ly -= g.n;
    if (lz < 0) lz += g.n;
}

constexpr int kRecPerThread = kBlockCap / kBlockThreads;
constexpr int kDenseB = 8;                    // an OWN cell with >= kDenseB records is DENSE: its same-cell pairs go to the tile role
constexpr int kMaxItems = (kBlockCap / kDenseB + 3) & ~3;  // (dense cell, tile) work items of one block
constexpr int kWarps = kBlockThreads / 32;
#ifndef FOF_QUEUE
#define FOF_QUEUE 256
#endif
constexpr int kQueue = FOF_QUEUE;                   // pairs a warp lists before it tests them
#ifndef FOF_LONGRUN
#define FOF_LONGRUN (1 << 30)  // off: measured slower (1.9 vs 1.2 ms at 256^3) than letting every lane list its own runs
#endif
constexpr int kLongRun = FOF_LONGRUN;                   // longer candidate runs are walked by the whole warp instead

struct BlockView {
    float4 *rec;          // [kBlockCap] records in local-cell order (x fastest)
    unsigned int *par;    // [kBlockCap] union-find parent (slot index)
    unsigned int *cbeg;   // [ncell + 1] first slot of every local cell
    unsigned int *items;  // [kMaxItems] cell | tile << 16
    unsigned int *queue;  // [kQueue] per warp: home slot << 16 | candidate slot
    int M;
};
__device__ __forceinline__ unsigned int lanemask_lt()
{
    unsigned int m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// ---- who tests which pair (every unordered pair in the same or in adjacent cells with at least one OWN end, once)
//   same cell, dense       the tile role: tiles of <= 32 records in registers, candidates broadcast, ballots;
//   everything else        the chunk role: the end whose cell sees the other one in its forward half stencil (+x; rows
//                          (dy, dz) = (+1, 0), (-1, +1), (0, +1), (+1, +1)) is the HOME of the pair and lists it.
// A pair (own, ghost) belongs to this block whatever its direction (no half space of cell offsets is consistent
// with the half space of block offsets), so a ghost is a home too, but lists OWN candidates only.

// =========================================================================================================
// chunk role: 32 consecutive slots, one home per lane.  Each home lists its candidate pairs into the warp's
// queue (runs of consecutive slots: a grid row of cells is contiguous), then all 32 lanes test listed pairs:
// a lane with forty candidates costs the others nothing.
// =========================================================================================================
template <bool WRAP>
__device__ __forceinline__ void chunk_role(const BlockView &v, int s0, const Grid &g, const BlockGeom &bg,
                                           const BlockOrigin &o, int lane, unsigned int &nedges, unsigned int &ntests)
{
    const float lo = g.reach, hi = 1.0f - g.reach;
    const int X = bg.X;
    const float4 *rec = v.rec;
    const unsigned int *cbeg = v.cbeg;
    const int s = s0 + lane;
    int b0 = 0, b1 = 0, b2 = 0, b3 = 0, b4 = 0, l0 = 0, l1 = 0, l2 = 0, l3 = 0, l4 = 0;  // run r = [b_r, b_r + l_r)
    float4 me = make_float4(0.f, 0.f, 0.f, 0.f);
    if (s < v.M) {
        me = rec[s];
        int lx, ly, lz;
        float fx, fy, fz;
        local_cell(me, g, bg, o, lx, ly, lz, fx, fy, fz);
        const int lc = lx + X * (ly + bg.Y * lz);
        const bool xl = fx < lo, xh = fx > hi, yl = fy < lo, yh = fy > hi, zh = fz > hi;
        // an own home meets every cell of the local grid; a ghost home meets OWN cells only (ghost-ghost pairs belong
        // to other blocks): rows ly' in [1, ncy], lz' < ncz, cells lx' in [1, ncx]
        const bool ghost = (__float_as_uint(me.w) & kGhostBit) != 0u;
        const int xmin = ghost ? 1 : 0, xmax = ghost ? o.ncx : X - 1;
        const int xa = max(lx - (xl ? 1 : 0), xmin), xb = min(lx + (xh ? 1 : 0), xmax);  // cells of a neighbour row
        auto row = [&](int dy, int dz, int &bb, int &ll) {
            const int yy = ly + dy, zz = lz + dz;
            if (xa > xb || (ghost && (yy < 1 || yy > o.ncy || zz >= o.ncz))) return;
            const int base = X * (yy + bg.Y * zz);
            bb = (int)cbeg[base + xa];
            ll = (int)cbeg[base + xb + 1] - bb;
        };
        const int c1 = (int)cbeg[lc + 1];
        if (!ghost) {
            // my cell after me (the tile role has the same-cell pairs of a dense cell) [+ the +x cell]
            b0 = c1 - (int)cbeg[lc] >= kDenseB ? c1 : s + 1;
            l0 = (xh ? (int)cbeg[lc + 2] : c1) - b0;
        } else if (xh && lx + 1 <= xmax && ly >= 1 && ly <= o.ncy && lz < o.ncz) {
            b0 = c1;
            l0 = (int)cbeg[lc + 2] - c1;
        }
        if (yh) row(1, 0, b1, l1);
        if (zh) {
            if (yl) row(-1, 1, b2, l2);
            row(0, 1, b3, l3);
            if (yh) row(1, 1, b4, l4);
        }
    }
    unsigned int *queue = v.queue;
    int nq = 0;  // pairs waiting in the queue (warp-uniform)
    auto drain = [&]() {
        __syncwarp();
        for (int q = lane; q < nq; q += 32) {  // the trip count differs by at most one between lanes
            const unsigned int e = queue[q];
            const int i = (int)(e >> 16), j = (int)(e & 0xffffu);
            if (linked_b<WRAP>(rec[i], rec[j], g)) {
                ++nedges;
                if (((volatile unsigned int *)v.par)[i] != ((volatile unsigned int *)v.par)[j]) unite_s(v.par, rec, i, j);
            }
        }
        __syncwarp();
        nq = 0;
    };
    // ---- long runs (a dense neighbour cell): listed by the whole warp, 32 pairs per pass
    if (__any_sync(kFull, max(max(max(l0, l1), max(l2, l3)), l4) >= kLongRun)) {
        auto long_runs = [&](int b, int &l) {
            unsigned int lng = __ballot_sync(kFull, l >= kLongRun);
            while (lng) {
                const int h = __ffs((int)lng) - 1;
                lng &= lng - 1u;
                const int bb = __shfl_sync(kFull, b, h), ll = __shfl_sync(kFull, l, h);
                const unsigned int hs = (unsigned int)(s0 + h) << 16;
                if (lane == 0) ntests += (unsigned int)ll;
                for (int off = 0; off < ll; off += 32) {
                    const int cnt = min(32, ll - off);
                    if (nq + cnt > kQueue) drain();
                    if (lane < cnt) queue[nq + lane] = hs | (unsigned int)(bb + off + lane);
                    nq += cnt;
                }
            }
            if (l >= kLongRun) l = 0;
        };
        long_runs(b0, l0); long_runs(b1, l1); long_runs(b2, l2); long_runs(b3, l3); long_runs(b4, l4);
    }
    // ---- short runs: each lane lists its own pairs behind what is already queued
    const int T = l0 + l1 + l2 + l3 + l4;
    int incl = T;
#pragma unroll
    for (int q = 1; q < 32; q <<= 1) {
        const int w = __shfl_up_sync(kFull, incl, q);
        if (lane >= q) incl += w;
    }
    const int total = __shfl_sync(kFull, incl, 31);
    if (total) {
        if (lane == 31) ntests += (unsigned int)total;
        const unsigned int hs = (unsigned int)s << 16;
        for (int w0 = 0; w0 < total;) {
            if (nq + min(total - w0, 32) > kQueue) drain();
            const int room = kQueue - nq;   // list the pairs at positions [w0, w0 + room) of the short list
            int base = incl - T - w0;       // position of my first pair relative to the window
            auto push = [&](int b, int l) {
                const int k0 = max(0, -base), k1 = min(l, room - base);
                for (int k = k0; k < k1; ++k) queue[nq + base + k] = hs | (unsigned int)(b + k);
                base += l;
            };
            push(b0, l0); push(b1, l1); push(b2, l2); push(b3, l3); push(b4, l4);
            const int n = min(room, total - w0);
            nq += n;
            w0 += n;
        }
    }
    if (nq) drain();
}

// =========================================================================================================
// tile role: the pairs inside one dense cell
// =========================================================================================================
// Returns, in lane k, the mask of tile lanes linked to the record at slot jb + k (k < cnt <= 32).
__device__ __forceinline__ unsigned int batch_adjacency_b(const float4 &me, const float4 *rec, int jb, int cnt,
                                                          const Grid &g, int lane)
{
    unsigned int adjT = 0;
#pragma unroll 4
    for (int k = 0; k < cnt; ++k) {
        const unsigned int bal = __ballot_sync(kFull, linked_b<false>(me, rec[jb + k], g));  // pairs inside one cell never wrap
        if (lane == k) adjT = bal;
    }
    return adjT;
}

__device__ __forceinline__ void tile_role(const BlockView &v, unsigned int item, const Grid &g, int lane,
                                          unsigned int &nedges, unsigned int &ntests)
{
    const float inf = __int_as_float(0x7f800000);
    const float4 *rec = v.rec;
    const int c = (int)(item & 0xffffu), t = (int)(item >> 16);
    const int d0 = (int)v.cbeg[c];
    const int m = (int)v.cbeg[c + 1] - d0;
    const int nt = (m + 31) >> 5, ts = (m + nt - 1) / nt;  // balanced tiles: 43 -> 22 + 21
    const int ib = d0 + t * ts;
    const int cntI = min(ts, m - t * ts);
    float4 me = make_float4(inf, inf, inf, 0.0f);  // a lane without a record sits at +inf: every test fails
    if (lane < cntI) me = rec[ib + lane];
    const unsigned int self = 1u << lane;
    // ---- the tile against itself
    const unsigned int adj = batch_adjacency_b(me, rec, ib, cntI, g, lane) & ~self;
    nedges += (unsigned int)__popc(adj & lanemask_lt());
    if (lane == 0) ntests += (unsigned int)(cntI * (cntI - 1) / 2);
    // components of the tile: breadth-first from the lowest unlabelled lane, one warp OR-reduction per level;
    // head = member with the smallest original index, every other member hooks straight under it
    unsigned int grp = self;
    int head = lane;
    if (__any_sync(kFull, adj != 0u)) {
        const unsigned int my_oi = lane < cntI ? (__float_as_uint(me.w) & ~kGhostBit) : 0xffffffffu;
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
            const unsigned int mn = __reduce_min_sync(kFull, in ? my_oi : 0xffffffffu);
            const unsigned int hb = __ballot_sync(kFull, in && my_oi == mn);
            if (in) { grp = vis; head = __ffs((int)hb) - 1; }
            todo &= ~vis;
        }
    }
    if (head != lane && atomicCAS(v.par + ib + lane, (unsigned int)(ib + lane), (unsigned int)(ib + head)) != (unsigned int)(ib + lane))
        unite_s(v.par, rec, ib + lane, ib + head);  // somebody hooked me first: general path
    __syncwarp();
    const bool leader = head == lane;
    // ---- the earlier tiles of my cell: candidate k (lane k's slot) joins every component of the tile it is linked to
    for (int jb = d0; jb < ib; jb += 32) {
        const int cnt = min(32, ib - jb);
        const unsigned int adjT = batch_adjacency_b(me, rec, jb, cnt, g, lane);
        nedges += (unsigned int)__popc(adjT);
        if (lane == 0) ntests += (unsigned int)(cnt * cntI);
        const unsigned int active = __reduce_or_sync(kFull, adjT);
        if (active) {
            unsigned int lead = __ballot_sync(kFull, leader && (grp & active));
            while (lead) {
                const int gl = __ffs((int)lead) - 1;
                lead &= lead - 1u;
                const unsigned int members = __shfl_sync(kFull, grp, gl);
                if (adjT & members) unite_s(v.par, rec, jb + lane, ib + gl);
            }
        }
        __syncwarp();
    }
}

template <bool WRAP>
__device__ __forceinline__ void link_phase(const BlockView &v, unsigned int nitems, unsigned int *ticket, const Grid &g,
                                           const BlockGeom &bg, const BlockOrigin &o, unsigned int &nedges,
                                           unsigned int &ntests)
{
    const int lane = (int)(threadIdx.x & 31u);
    const unsigned int nchunks = (unsigned int)((v.M + 31) >> 5);
    while (true) {  // warps draw tiles first (the long items), then chunks
        unsigned int it = 0;
        if (lane == 0) it = atomicAdd(ticket, 1u);
        it = __shfl_sync(kFull, it, 0);
        DBG_T(t0);
#ifdef FOF_ABL_NOTILE
        if (it < nitems) { }
#else
        if (it < nitems) { tile_role(v, v.items[it], g, lane, nedges, ntests); DBG_T(t1); DBG_ADD(4, t0, t1); DBG_ADD(8, 0, 1); }
#endif
#ifdef FOF_ABL_NOCHUNK
        else if (it - nitems < nchunks) { }
#else
        else if (it - nitems < nchunks) { chunk_role<WRAP>(v, (int)(it - nitems) * 32, g, bg, o, lane, nedges, ntests); DBG_T(t1); DBG_ADD(5, t0, t1); DBG_ADD(9, 0, 1); }
#endif
        else break;
    }
}

__global__ void __launch_bounds__(kBlockThreads, 2) block_link_kernel(const float4 *__restrict__ part,
                                                                      const unsigned int *__restrict__ cursor,
                                                                      unsigned int cap, Grid g, BlockGeom bg, int *labels,
                                                                      int2 *__restrict__ cross, unsigned int cross_cap,
                                                                      Ctrl *ctrl)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    BlockView v;
    v.rec = reinterpret_cast<float4 *>(smem_raw);
    v.par = reinterpret_cast<unsigned int *>(smem_raw + (size_t)kBlockCap * 16);
    v.items = v.par + kBlockCap;
    v.queue = v.items + kMaxItems + kQueue * (threadIdx.x >> 5);
    v.cbeg = v.items + kMaxItems + kQueue * kWarps;  // [ncell + 1]
    __shared__ unsigned long long s_bar;
    __shared__ unsigned int s_warp[kWarps];
    __shared__ unsigned int s_red[2], s_nitems, s_ticket;
    if (*(volatile unsigned int *)&ctrl->mode) return;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const size_t p0 = (size_t)blockIdx.x * cap;
    const int M = (int)cursor[blockIdx.x];  // <= cap: an overflowing block has set ctrl->mode
    if (M == 0) return;
    float4 *rec = v.rec;
    unsigned int *cbeg = v.cbeg;
    v.M = M;
    DBG_T(tA);

    // ---- A: one TMA bulk copy brings the block's records in; meanwhile the cell counters are cleared
    if (tid == 0) {
        mbar_init(&s_bar, 1);
        mbar_expect_tx(&s_bar, (unsigned int)M * 16u);
        tma_load_1d(rec, part + p0, (unsigned int)M * 16u, &s_bar);
        s_red[0] = s_red[1] = 0u;
        s_nitems = 0u;
        s_ticket = 0u;
        if ((unsigned int)M > *(volatile unsigned int *)&ctrl->max_block) atomicMax(&ctrl->max_block, (unsigned int)M);
    }
    const int ncell = bg.ncell;
    for (int c = tid; c <= ncell; c += kBlockThreads) cbeg[c] = 0u;
    BlockOrigin o;
    {
        const int b = blockIdx.x;
        const int bx = b % bg.nbx, by = (b / bg.nbx) % bg.nby, bz = b / (bg.nbx * bg.nby);
        o.x0 = bx << bg.sx; o.y0 = by << bg.sy; o.z0 = bz << bg.sz;
        o.ncx = min(1 << bg.sx, g.n - o.x0); o.ncy = min(1 << bg.sy, g.n - o.y0); o.ncz = min(1 << bg.sz, g.n - o.z0);
    }
    // pairs of this block can cross a box face only if the block touches one
    const bool wrap = o.x0 == 0 || o.y0 == 0 || o.x0 + (1 << bg.sx) >= g.n || o.y0 + (1 << bg.sy) >= g.n ||
                      o.z0 + (1 << bg.sz) >= g.n;
    __syncthreads();
    mbar_wait(&s_bar, 0);
    DBG_T(tB);
    DBG_ADD(0, tA, tB);

    // ---- B: counting sort by local cell, in place (records pass through registers)
    float4 r[kRecPerThread];
    unsigned int key[kRecPerThread];  // local cell << 16 | rank inside the cell
#pragma unroll
    for (int k = 0; k < kRecPerThread; ++k) {
        const int s = tid + k * kBlockThreads;
        if (s < M) {
            r[k] = rec[s];
            int lx, ly, lz;
            float fx, fy, fz;
            local_cell(r[k], g, bg, o, lx, ly, lz, fx, fy, fz);
            const int lc = lx + bg.X * (ly + bg.Y * lz);
            key[k] = ((unsigned int)lc << 16) | atomicAdd(&cbeg[lc], 1u);
        }
    }
    __syncthreads();
    {   // exclusive scan of the cell counts: thread t owns cells [t per, (t + 1) per)
        const int per = (ncell + kBlockThreads - 1) / kBlockThreads;
        const int c0 = min(tid * per, ncell), c1 = min(c0 + per, ncell);
        unsigned int sum = 0;
        for (int c = c0; c < c1; ++c) sum += cbeg[c];
        unsigned int incl = sum;
#pragma unroll
        for (int q = 1; q < 32; q <<= 1) {
            const unsigned int t = __shfl_up_sync(kFull, incl, q);
            if (lane >= q) incl += t;
        }
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        unsigned int woff = 0;
#pragma unroll
        for (int w = 0; w < kWarps; ++w)
            if (w < warp) woff += s_warp[w];
        unsigned int run = woff + incl - sum;
        for (int c = c0; c < c1; ++c) {
            const unsigned int n = cbeg[c];
            cbeg[c] = run;
            run += n;
            if (n >= (unsigned int)kDenseB) {  // a dense OWN cell: one work item per tile of <= 32 records
                const int lx = c % bg.X, ly = (c / bg.X) % bg.Y, lz = c / (bg.X * bg.Y);
                if (lx >= 1 && lx <= o.ncx && ly >= 1 && ly <= o.ncy && lz < o.ncz) {
                    const unsigned int nt = (n + 31u) >> 5;
                    const unsigned int at = atomicAdd(&s_nitems, nt);
                    for (unsigned int t = 0; t < nt; ++t) v.items[at + t] = (unsigned int)c | (t << 16);
                }
            }
        }
        if (tid == 0) cbeg[ncell] = (unsigned int)M;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < kRecPerThread; ++k) {
        const int s = tid + k * kBlockThreads;
        if (s < M) {
            const int slot = (int)(cbeg[key[k] >> 16] + (key[k] & 0xffffu));
            rec[slot] = r[k];
            v.par[slot] = (unsigned int)slot;
        }
    }
    __syncthreads();

    DBG_T(tC);
    DBG_ADD(1, tB, tC);
    // ---- C: pair tests + unions
    unsigned int nedges = 0, ntests = 0;
    if (wrap) link_phase<true>(v, s_nitems, &s_ticket, g, bg, o, nedges, ntests);
    else link_phase<false>(v, s_nitems, &s_ticket, g, bg, o, nedges, ntests);
    DBG_T(tC2);
    DBG_ADD(6, tC, tC2);
    __syncthreads();
    DBG_T(tD);
    DBG_ADD(2, tC, tD);

    // ---- D: labels of my own non-roots; one equivalence per linked ghost
    for (int s0 = warp * 32; s0 < M; s0 += kBlockThreads) {
        const int s = s0 + lane;
        bool emit = false;
        unsigned int me_o = 0, root_o = 0;
        if (s < M) {
            const int rt = find_s(v.par, s);
            if (rt != s) {
                const unsigned int w = __float_as_uint(rec[s].w);
                me_o = w & ~kGhostBit;
                root_o = orig_of(rec, rt);
                if (w & kGhostBit) emit = true;
                else labels[me_o] = (int)root_o;
            }
        }
        const unsigned int bal = __ballot_sync(kFull, emit);
        if (bal) {
            unsigned int at = 0;
            if (lane == 0) at = atomicAdd(&ctrl->ncross, (unsigned int)__popc(bal));
            at = __shfl_sync(kFull, at, 0);
            if (emit) {
                const unsigned int k = at + (unsigned int)__popc(bal & ((1u << lane) - 1u));
                if (k < cross_cap) cross[k] = make_int2((int)me_o, (int)root_o);
                else ctrl->mode = 1u;  // more linked ghosts than the list holds (tiny blocks): the cell path takes over --
                                       // it rewrites labels and counters from scratch, so what this kernel wrote is moot
            }
        }
    }
    nedges = __reduce_add_sync(kFull, nedges);
    ntests = __reduce_add_sync(kFull, ntests);
    if (lane == 0) { atomicAdd(&s_red[0], nedges); atomicAdd(&s_red[1], ntests); }
    __syncthreads();
    DBG_T(tE);
    DBG_ADD(3, tD, tE);
    if (tid == 0) {
        if (s_red[0]) atomicAdd(&ctrl->edges_b, (unsigned long long)s_red[0]);
        if (s_red[1]) atomicAdd(&ctrl->pair_tests_b, (unsigned long long)s_red[1]);
    }
}

// ---------------------------------------------------------------------------------------------------------
// global union-find on `labels` (parent = original index, labels[r] == r at a root, parent < child)
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ int find_g(int *lab, int x)
{
    int p = ((volatile int *)lab)[x];
    while (p != x) {
        const int gp = ((volatile int *)lab)[p];
        if (gp != p) ((volatile int *)lab)[x] = gp;
        x = p;
        p = gp;
    }
    return x;
}

__global__ void __launch_bounds__(kBlock) cross_link_kernel(const int2 *__restrict__ cross, int *labels, Ctrl *ctrl)
{
    if (*(volatile unsigned int *)&ctrl->mode) return;
    const unsigned int n = *(volatile unsigned int *)&ctrl->ncross;  // <= the list's capacity, or mode is set
    for (unsigned int k = blockIdx.x * kBlock + threadIdx.x; k < n; k += gridDim.x * kBlock) {
        const int2 e = cross[k];
        int ra = find_g(labels, e.x), rb = find_g(labels, e.y);
        while (ra != rb) {
            if (ra < rb) { const int t = ra; ra = rb; rb = t; }  // ra: larger index, hooks under rb
            const int old = atomicCAS(labels + ra, ra, rb);
            if (old == ra) break;
            ra = find_g(labels, old);
        }
    }
}

// labels[i] = root(i); four particles per thread.  Only the thread that owns i writes labels[i]; what it reads
// of other entries is the parent or an ancestor, old or new.
__global__ void __launch_bounds__(kBlock) flatten_labels_kernel(int *labels, int64_t N, bool vec, Ctrl *ctrl,
                                                                int *__restrict__ cnt, unsigned long long *state,
                                                                int64_t state_items)
{
    if (*(volatile const unsigned int *)&ctrl->mode) return;
    {   // H6 rides along (see write_labels_kernel): clear the state of the compaction scan of fof_groups
        const int64_t tid = (int64_t)blockIdx.x * kBlock + threadIdx.x;
        if (tid == 0) { ctrl->gscan_ticket = 0u; ctrl->K = 0; }
        for (int64_t k = tid; k < state_items; k += (int64_t)gridDim.x * kBlock) state[k] = 0ull;
    }
    const int64_t i0 = ((int64_t)blockIdx.x * kBlock + threadIdx.x) * 4;
    if (i0 >= N) return;
    int l[4];
    if (vec && i0 + 4 <= N) {
        const int4 t = *reinterpret_cast<const int4 *>(labels + i0);
        l[0] = t.x; l[1] = t.y; l[2] = t.z; l[3] = t.w;
    } else {
#pragma unroll
        for (int k = 0; k < 4; ++k) l[k] = i0 + k < N ? labels[i0 + k] : (int)(i0 + k);
    }
    bool any = false;
#pragma unroll
    for (int k = 0; k < 4; ++k) any |= l[k] != (int)(i0 + k);
    if (!any) return;
    int r[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) r[k] = l[k];
    bool moving = true;
    while (moving) {
        int p[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) p[k] = i0 + k < N ? ((volatile int *)labels)[r[k]] : r[k];  // nothing to chase behind the last particle
        moving = false;
#pragma unroll
        for (int k = 0; k < 4; ++k) { moving |= p[k] != r[k]; r[k] = p[k]; }
    }
#pragma unroll
    for (int k = 0; k < 4; ++k)
        if (i0 + k < N && r[k] != (int)(i0 + k)) {  // a non-root: one more member of r[k]'s group
            if (r[k] != l[k]) labels[i0 + k] = r[k];
            atomicAdd(cnt + r[k], 1);
        }
}

inline size_t block_link_smem(const BlockGeom &bg)
{
    return (size_t)kBlockCap * 20 + (size_t)kMaxItems * 4 + (size_t)kWarps * kQueue * 4 + ((size_t)bg.ncell + 1) * 4;
}

inline cudaError_t set_smem(const void *fn, size_t bytes)
{
    if (bytes <= 40 * 1024) return cudaSuccess;  // static shared memory counts against the 48 KB default too
    return cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

}  // namespace

#ifdef FOF_BLOCK_TIMING
extern "C" void fof_dbg_read(unsigned long long *out, int reset)
{
    cudaMemcpyFromSymbol(out, g_dbg, sizeof(g_dbg));
    if (reset) { unsigned long long z[16] = {0}; cudaMemcpyToSymbol(g_dbg, z, sizeof(z)); }
}
#endif

cudaError_t launch_block_path(const float *pos, int64_t N, Grid g, const BlockGeom &bg, int ctas, unsigned int *cursor,
                              float4 *part, int2 *cross, int *labels, int *cnt, unsigned long long *state,
                              int64_t state_items, Ctrl *ctrl, StageHook &hook, cudaStream_t s)
{
    if (N <= 0) return cudaSuccess;
    cudaError_t e;
    const bool vec = ((uintptr_t)pos & 15) == 0;
    const bool labels_vec = ((uintptr_t)labels & 15) == 0;
    const size_t smem_bins = (size_t)bg.bins * sizeof(unsigned int);
    const size_t smem_link = block_link_smem(bg);
    auto scat = vec ? block_scatter_kernel<true> : block_scatter_kernel<false>;
    if ((e = set_smem((const void *)scat, smem_bins)) != cudaSuccess) return e;
    if ((e = set_smem((const void *)block_link_kernel, smem_link)) != cudaSuccess) return e;
    hook.begin(0, 1);
    if ((e = cudaMemsetAsync(cursor, 0, smem_bins, s)) != cudaSuccess) return e;
    scat<<<FOF_SCAT_CTAS * ctas, kScatThreads, smem_bins, s>>>(pos, N, g, bg, cursor, part, (unsigned int)kBlockCap, labels,
                                                              labels_vec, cnt, ctrl);
    hook.end(0);
    hook.begin(1, 1);
    block_link_kernel<<<bg.bins, kBlockThreads, smem_link, s>>>(part, cursor, (unsigned int)kBlockCap, g, bg, labels, cross,
                                                                (unsigned int)(N + 1), ctrl);
    hook.end(1);
    hook.begin(2, 1);
    cross_link_kernel<<<2 * ctas, kBlock, 0, s>>>(cross, labels, ctrl);
    hook.end(2);
    hook.begin(3, 1);
    flatten_labels_kernel<<<(unsigned int)((N + 4 * kBlock - 1) / (4 * kBlock)), kBlock, 0, s>>>(labels, N, labels_vec, ctrl, cnt, state,
                                                                                                 state_items);
    hook.end(3);
    return cudaGetLastError();
}

}  // namespace fof
