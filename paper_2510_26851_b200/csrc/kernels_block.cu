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
//   block_hist_kernel     records (own + ghost) per block                        pos -> bin_total
//   block_offsets_kernel  exclusive scan; decides ctrl->mode (1 = a block does not fit: cell path runs)
//   block_scatter_kernel  records to their blocks through shared cursors          pos -> part, labels[i] = i
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
// records per block: per-CTA histogram in shared memory, then one global atomic per (CTA, non-empty block)
// ---------------------------------------------------------------------------------------------------------
template <bool VEC>
__global__ void __launch_bounds__(kPartThreads) block_hist_kernel(const float *__restrict__ pos, int64_t N, Grid g,
                                                                  BlockGeom bg, int64_t chunk,
                                                                  unsigned int *__restrict__ bin_total, Ctrl *ctrl)
{
    extern __shared__ unsigned int s_bin[];
    for (int b = threadIdx.x; b < bg.bins; b += kPartThreads) s_bin[b] = 0u;
    __syncthreads();
    const int64_t i0 = (int64_t)blockIdx.x * chunk;
    const int64_t i1 = min(N, i0 + chunk);
    bool bad = false;
    for_each_particle<VEC, kPartThreads>(pos, i0, i1, [&](float x, float y, float z, int64_t) {
        wrap3(x, y, z, g, bad);
        const unsigned int own = classify(x, y, z, g, bg, [&](unsigned int gb) { atomicAdd(&s_bin[gb], 1u); });
        atomicAdd(&s_bin[own], 1u);
    });
    if (bad) atomicOr(&ctrl->error, 1u);
    __syncthreads();
    for (int b = threadIdx.x; b < bg.bins; b += kPartThreads) {
        const unsigned int c = s_bin[b];
        if (c) atomicAdd(&bin_total[b], c);
    }
}

// ---------------------------------------------------------------------------------------------------------
// one CTA: exclusive scan of the block totals -> bin_base (and the write cursors), fullest block, mode
// ---------------------------------------------------------------------------------------------------------
constexpr int kOffThreads = 1024;
__global__ void __launch_bounds__(kOffThreads) block_offsets_kernel(const unsigned int *__restrict__ bin_total, int bins,
                                                                    unsigned int *__restrict__ bin_base,
                                                                    unsigned int *__restrict__ cursor, unsigned int cap,
                                                                    unsigned long long part_cap, Ctrl *ctrl)
{
    __shared__ unsigned int s_warp[kOffThreads / 32];
    __shared__ unsigned int s_max[kOffThreads / 32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int per = (bins + kOffThreads - 1) / kOffThreads;
    const int b0 = tid * per, b1 = min(bins, b0 + per);
    unsigned int sum = 0, mx = 0;
    for (int b = b0; b < b1; ++b) { const unsigned int c = bin_total[b]; sum += c; mx = max(mx, c); }
    unsigned int incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned int t = __shfl_up_sync(kFull, incl, o);
        if (lane >= o) incl += t;
    }
    mx = __reduce_max_sync(kFull, mx);
    if (lane == 31) s_warp[warp] = incl;
    if (lane == 0) s_max[warp] = mx;
    __syncthreads();
    unsigned int woff = 0, total = 0, gmax = 0;
#pragma unroll
    for (int w = 0; w < kOffThreads / 32; ++w) {
        const unsigned int t = s_warp[w];
        if (w < warp) woff += t;
        total += t;
        gmax = max(gmax, s_max[w]);
    }
    unsigned int run = woff + incl - sum;
    for (int b = b0; b < b1; ++b) {
        bin_base[b] = run;
        cursor[b] = run;
        run += bin_total[b];
    }
    if (tid == 0) {
        bin_base[bins] = total;
        ctrl->max_block = gmax;
        ctrl->mode = (gmax > cap || (unsigned long long)total > part_cap) ? 1u : 0u;
    }
}

// ---------------------------------------------------------------------------------------------------------
// records to their blocks.  A CTA takes tiles of TH x PER particles (registers); the rank of a record among
// the tile's records of its block comes from a shared-memory counter, the tile's slice of the block from ONE
// global atomic per (tile, non-empty block) on the block's cursor: all CTAs append to the same few thousand
// open lines, which the L2 merges before they reach DRAM (private per-CTA streams: 0.42 ms, shared: 0.25 ms for
// 2^24 records into 4096 blocks).  The rare ghost copies take one global atomic each.
// ---------------------------------------------------------------------------------------------------------
constexpr int kScatThreads = 512, kScatPer = 8;

template <bool VEC>
__global__ void __launch_bounds__(kScatThreads) block_scatter_kernel(const float *__restrict__ pos, int64_t N, Grid g,
                                                                     BlockGeom bg, unsigned int *cursor,
                                                                     float4 *__restrict__ part, int *__restrict__ labels,
                                                                     bool labels_vec, Ctrl *ctrl)
{
    extern __shared__ unsigned int s_cnt[];  // [bins]
    __shared__ unsigned int s_tile;
    if (*(volatile unsigned int *)&ctrl->mode) return;
    constexpr int T = kScatThreads * kScatPer;
    const int64_t ntiles = (N + T - 1) / T;
    const int tid = threadIdx.x;
    for (;;) {
        __syncthreads();
        if (tid == 0) s_tile = atomicAdd(&ctrl->tile_ticket2, 1u);
        for (int b = tid; b < bg.bins; b += kScatThreads) s_cnt[b] = 0u;
        __syncthreads();
        const int64_t tile = s_tile;
        if (tile >= ntiles) return;
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
            // H5, first half: labels[i] = i (final for every singleton), coalesced
            if (labels_vec && i + 4 <= N) *reinterpret_cast<int4 *>(labels + i) = make_int4((int)i, (int)i + 1, (int)i + 2, (int)i + 3);
            else
                for (int k = 0; k < 4; ++k) if (i + k < N) labels[i + k] = (int)(i + k);
        }
        bool bad = false;
#pragma unroll
        for (int k = 0; k < kScatPer; ++k) {
            bin[k] = 0xffffffffu;
            if (__float_as_int(rec[k].w) >= 0) {
                wrap3(rec[k].x, rec[k].y, rec[k].z, g, bad);
                const float4 r = rec[k];
                bin[k] = classify(r.x, r.y, r.z, g, bg, [&](unsigned int gb) {
                    part[atomicAdd(&cursor[gb], 1u)] =
                        make_float4(r.x, r.y, r.z, __uint_as_float(__float_as_uint(r.w) | kGhostBit));
                });
                rank[k] = atomicAdd(&s_cnt[bin[k]], 1u);
            }
        }
        __syncthreads();
        for (int b = tid; b < bg.bins; b += kScatThreads) {
            const unsigned int c = s_cnt[b];
            if (c) s_cnt[b] = atomicAdd(&cursor[b], c);
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < kScatPer; ++k)
            if (bin[k] != 0xffffffffu) part[s_cnt[bin[k]] + rank[k]] = rec[k];
    }
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

// Every pair (own, own) in the same or in adjacent cells is tested by the particle whose cell sees the other
// one in its forward half stencil (+x, then the rows (dy, dz) = (+1, 0), (-1, +1), (0, +1), (+1, +1)); a row is
// one contiguous run of slots (x-fastest local cell ids), trimmed to the cells the home particle can reach.
// A pair (own, ghost) belongs to this block whatever its direction, so a ghost is a home particle too, but
// only against OWN candidates (ghost-ghost pairs belong to other blocks).
template <bool WRAP>
__device__ __forceinline__ void link_phase(const float4 *rec, const unsigned int *cbeg, unsigned int *par, int M,
                                           const Grid &g, const BlockGeom &bg, const BlockOrigin &o,
                                           unsigned int &nedges, unsigned int &ntests)
{
    const float lo = g.reach, hi = 1.0f - g.reach;
    const int X = bg.X, XY = bg.X * bg.Y;
    const int lane = (int)(threadIdx.x & 31u);
    // One home particle per lane; its (up to five) candidate runs are walked as ONE list, all lanes of the warp
    // in lock step (warp-uniform trip count, __syncwarp() per trip: left to themselves the lanes drift apart
    // through the unions and never reconverge -- measured 3 of 32 lanes active).
    for (int s0 = (int)(threadIdx.x & ~31u); s0 < M; s0 += kBlockThreads) {
        const int s = s0 + lane;
        int b0 = 0, b1 = 0, b2 = 0, b3 = 0, b4 = 0, e0 = 0, e1 = 0, e2 = 0, e3 = 0, e4 = 0;  // run r = [b_r, b_r + len_r); e_r = prefix ends
        float4 me = make_float4(0.f, 0.f, 0.f, 0.f);
        if (s < M) {
            me = rec[s];
            int lx, ly, lz;
            float fx, fy, fz;
            local_cell(me, g, bg, o, lx, ly, lz, fx, fy, fz);
            const int lc = lx + X * (ly + bg.Y * lz);
            const bool xl = fx < lo, xh = fx > hi, yl = fy < lo, yh = fy > hi, zh = fz > hi;
            const int ol = xl ? 1 : 0, oh = xh ? 1 : 0;
            if (!(__float_as_uint(me.w) & kGhostBit)) {
                b0 = s + 1; e0 = (int)cbeg[lc + 1 + oh] - b0;  // my cell after me [+ the +x cell]
                if (yh) { b1 = (int)cbeg[lc + X - ol]; e1 = (int)cbeg[lc + X + 1 + oh] - b1; }
                if (zh) {
                    const int up = lc + XY;
                    if (yl) { b2 = (int)cbeg[up - X - ol]; e2 = (int)cbeg[up - X + 1 + oh] - b2; }
                    b3 = (int)cbeg[up - ol]; e3 = (int)cbeg[up + 1 + oh] - b3;
                    if (yh) { b4 = (int)cbeg[up + X - ol]; e4 = (int)cbeg[up + X + 1 + oh] - b4; }
                }
            } else {
                // a ghost meets OWN cells only: row (ly + dy, lz + dz), cells lx + xa .. lx + xb clipped to [1, ncx]
                auto row = [&](int dy, int dz, int xa, int xb, int &bb, int &ll) {
                    const int yy = ly + dy, zz = lz + dz;
                    if (yy < 1 || yy > o.ncy || zz >= o.ncz) return;
                    const int a = max(lx + xa, 1), b = min(lx + xb, o.ncx);
                    if (a > b) return;
                    const int base = X * (yy + bg.Y * zz);
                    bb = (int)cbeg[base + a];
                    ll = (int)cbeg[base + b + 1] - bb;
                };
                if (xh) row(0, 0, 1, 1, b0, e0);
                if (yh) row(1, 0, -ol, oh, b1, e1);
                if (zh) {
                    if (yl) row(-1, 1, -ol, oh, b2, e2);
                    row(0, 1, -ol, oh, b3, e3);
                    if (yh) row(1, 1, -ol, oh, b4, e4);
                }
            }
        }
        // prefix ends; run r covers list positions [e_{r-1}, e_r)
        e1 += e0; e2 += e1; e3 += e2; e4 += e3;
        ntests += (unsigned int)e4;
        const int trips = __reduce_max_sync(kFull, e4);
        int ri = s;  // a slot known to be in my set (skips the union when the partner already points at it)
        for (int k = 0; k < trips; ++k) {
            if (k < e4) {
                const int j = k < e0 ? b0 + k : (k < e1 ? b1 + (k - e0) : (k < e2 ? b2 + (k - e1) : (k < e3 ? b3 + (k - e2) : b4 + (k - e3))));
                if (linked_b<WRAP>(me, rec[j], g)) {
                    ++nedges;
                    if ((int)((volatile unsigned int *)par)[j] != ri) ri = unite_s(par, rec, s, j);
                }
            }
            __syncwarp();
        }
    }
}

__global__ void __launch_bounds__(kBlockThreads, 2) block_link_kernel(const float4 *__restrict__ part,
                                                                      const unsigned int *__restrict__ bin_base, Grid g,
                                                                      BlockGeom bg, int *labels, int2 *__restrict__ cross,
                                                                      Ctrl *ctrl)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float4 *rec = reinterpret_cast<float4 *>(smem_raw);                                  // [kBlockCap]
    unsigned int *par = reinterpret_cast<unsigned int *>(smem_raw + (size_t)kBlockCap * 16);  // [kBlockCap]
    unsigned int *cbeg = par + kBlockCap;                                                // [ncell + 1]
    __shared__ unsigned long long s_bar;
    __shared__ unsigned int s_warp[kBlockThreads / 32];
    __shared__ unsigned int s_red[2];
    if (*(volatile unsigned int *)&ctrl->mode) return;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned int p0 = bin_base[blockIdx.x];
    const int M = (int)(bin_base[blockIdx.x + 1] - p0);
    if (M == 0) return;

    // ---- A: one TMA bulk copy brings the block's records in; meanwhile the cell counters are cleared
    if (tid == 0) {
        mbar_init(&s_bar, 1);
        mbar_expect_tx(&s_bar, (unsigned int)M * 16u);
        tma_load_1d(rec, part + p0, (unsigned int)M * 16u, &s_bar);
        s_red[0] = s_red[1] = 0u;
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
        for (int w = 0; w < kBlockThreads / 32; ++w)
            if (w < warp) woff += s_warp[w];
        unsigned int run = woff + incl - sum;
        for (int c = c0; c < c1; ++c) { const unsigned int t = cbeg[c]; cbeg[c] = run; run += t; }
        if (tid == 0) cbeg[ncell] = (unsigned int)M;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < kRecPerThread; ++k) {
        const int s = tid + k * kBlockThreads;
        if (s < M) {
            const int slot = (int)(cbeg[key[k] >> 16] + (key[k] & 0xffffu));
            rec[slot] = r[k];
            par[slot] = (unsigned int)slot;
        }
    }
    __syncthreads();

    // ---- C: half-stencil tests + unions
    unsigned int nedges = 0, ntests = 0;
    if (wrap) link_phase<true>(rec, cbeg, par, M, g, bg, o, nedges, ntests);
    else link_phase<false>(rec, cbeg, par, M, g, bg, o, nedges, ntests);
    __syncthreads();

    // ---- D: labels of my own non-roots; one equivalence per linked ghost
    for (int s0 = warp * 32; s0 < M; s0 += kBlockThreads) {
        const int s = s0 + lane;
        bool emit = false;
        unsigned int me_o = 0, root_o = 0;
        if (s < M) {
            const int rt = find_s(par, s);
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
            if (emit) cross[at + __popc(bal & ((1u << lane) - 1u))] = make_int2((int)me_o, (int)root_o);
        }
    }
    nedges = __reduce_add_sync(kFull, nedges);
    ntests = __reduce_add_sync(kFull, ntests);
    if (lane == 0) { atomicAdd(&s_red[0], nedges); atomicAdd(&s_red[1], ntests); }
    __syncthreads();
    if (tid == 0) {
        if (s_red[0]) atomicAdd(&ctrl->edges, (unsigned long long)s_red[0]);
        if (s_red[1]) atomicAdd(&ctrl->pair_tests, (unsigned long long)s_red[1]);
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
    const unsigned int n = *(volatile unsigned int *)&ctrl->ncross;
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
__global__ void __launch_bounds__(kBlock) flatten_labels_kernel(int *labels, int64_t N, bool vec, const Ctrl *ctrl)
{
    if (*(volatile const unsigned int *)&ctrl->mode) return;
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
        for (int k = 0; k < 4; ++k) p[k] = ((volatile int *)labels)[r[k]];
        moving = false;
#pragma unroll
        for (int k = 0; k < 4; ++k) { moving |= p[k] != r[k]; r[k] = p[k]; }
    }
#pragma unroll
    for (int k = 0; k < 4; ++k)
        if (i0 + k < N && r[k] != l[k]) labels[i0 + k] = r[k];
}

inline cudaError_t set_smem(const void *fn, size_t bytes)
{
    if (bytes <= 48 * 1024) return cudaSuccess;
    return cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

}  // namespace

cudaError_t launch_block_path(const float *pos, int64_t N, Grid g, const BlockGeom &bg, int ctas, unsigned int *bin_total,
                              unsigned int *bin_base, unsigned int *cursor, float4 *part, int64_t part_cap, int2 *cross,
                              int *labels, Ctrl *ctrl, StageHook &hook, cudaStream_t s)
{
    if (N <= 0) return cudaSuccess;
    cudaError_t e;
    const bool vec = ((uintptr_t)pos & 15) == 0;
    const bool labels_vec = ((uintptr_t)labels & 15) == 0;
    const size_t smem_bins = (size_t)bg.bins * sizeof(unsigned int);
    const size_t smem_link = (size_t)kBlockCap * 20 + ((size_t)bg.ncell + 1) * sizeof(unsigned int);
    auto hist = vec ? block_hist_kernel<true> : block_hist_kernel<false>;
    auto scat = vec ? block_scatter_kernel<true> : block_scatter_kernel<false>;
    if ((e = set_smem((const void *)hist, smem_bins)) != cudaSuccess) return e;
    if ((e = set_smem((const void *)scat, smem_bins)) != cudaSuccess) return e;
    if ((e = set_smem((const void *)block_link_kernel, smem_link)) != cudaSuccess) return e;
    const int64_t chunk = ((N + ctas - 1) / ctas + 3) & ~(int64_t)3;
    hook.begin(0, 1);
    if ((e = cudaMemsetAsync(bin_total, 0, smem_bins, s)) != cudaSuccess) return e;
    hist<<<ctas, kPartThreads, smem_bins, s>>>(pos, N, g, bg, chunk, bin_total, ctrl);
    hook.end(0);
    hook.begin(1, 1);
    block_offsets_kernel<<<1, kOffThreads, 0, s>>>(bin_total, bg.bins, bin_base, cursor, (unsigned int)kBlockCap,
                                                   (unsigned long long)part_cap, ctrl);
    hook.end(1);
    hook.begin(2, 1);
    scat<<<2 * ctas, kScatThreads, smem_bins, s>>>(pos, N, g, bg, cursor, part, labels, labels_vec, ctrl);
    hook.end(2);
    hook.begin(3, 1);
    block_link_kernel<<<bg.bins, kBlockThreads, smem_link, s>>>(part, bin_base, g, bg, labels, cross, ctrl);
    hook.end(3);
    hook.begin(4, 1);
    cross_link_kernel<<<2 * ctas, kBlock, 0, s>>>(cross, labels, ctrl);
    hook.end(4);
    hook.begin(5, 1);
    flatten_labels_kernel<<<(unsigned int)((N + 4 * kBlock - 1) / (4 * kBlock)), kBlock, 0, s>>>(labels, N, labels_vec, ctrl);
    hook.end(5);
    return cudaGetLastError();
}

}  // namespace fof
