// kernels_subhalo.cu — six-dimensional sub-halo pass.
// PAPER.md:141-154 (section 2.1.1): "For each identified halo, we then collect the particles
// associated with it and rerun a second FoF pass" in phase space with the metric of Eq. 3,
//     d(i,j)^2 = (x_i - x_j)^2 / sigma_x + (v_i - v_j)^2 / sigma_v.
// Readings R29-R31 of DESIGN.md: float32 predicate without FMA, d2 <= ell2; labels = minimum original
// index of the 6-D component inside one kept halo; particles of dropped halos keep their own index.
// Steps: member lists per halo (exclusive scan of the group sizes, atomic fill), all pairs inside
// each halo tile by tile (one warp per tile of 32 members, the partner tile staged
// in shared memory), lock-free union-find over member slots ordered by original index, labels.
// Cost is O(sum of squared halo sizes): meant for halos, not for a percolating component.
#include "fof_internal.cuh"

namespace fof {

struct Sub6 {
    float L, h, rx, rv, ell2;
};

constexpr int kSubSmall = 256;  // halos up to this many members: one warp each
constexpr int kSubChunk = 16;   // partner tiles per work item of a larger halo

// Work items of a halo of T tiles: tile row `it` has it / kSubChunk + 1 chunks of partner tiles.
__host__ __device__ __forceinline__ unsigned long long sub_items(unsigned int M)
{
    if (M <= (unsigned int)kSubSmall) return 0ull;
    const unsigned long long T = (M + 31u) >> 5, q = T / kSubChunk, r = T % kSubChunk;
    return (unsigned long long)kSubChunk * (q * (q + 1ull) / 2ull) + r * (q + 1ull);
}

// offsets[k] = sum of group_size[0..k), offsets[K] = number of members; cursor[k] = 0;
// work_off[k] = sum of sub_items(group_size[0..k)), work_off[K] = number of work items.
// Two launches over chunks of kSubScan halos: the totals of every chunk, then each CTA adds up the
// totals before its chunk and scans the chunk.
constexpr int kSubPer = 8, kSubScan = 1024 * kSubPer;

struct SubTotal {
    unsigned long long items;
    unsigned long long members;
};

__device__ __forceinline__ SubTotal sub_block_sum(unsigned long long members, unsigned long long items)
{
    __shared__ unsigned long long s_m[32], s_w[32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int o = 16; o > 0; o >>= 1) {
        members += __shfl_xor_sync(0xffffffffu, members, o);
        items += __shfl_xor_sync(0xffffffffu, items, o);
    }
    if (lane == 0) { s_m[warp] = members; s_w[warp] = items; }
    __syncthreads();
    SubTotal t = {0ull, 0ull};
    for (int w = 0; w < 32; ++w) { t.members += s_m[w]; t.items += s_w[w]; }
    __syncthreads();
    return t;
}

__global__ void __launch_bounds__(1024) sub_totals_kernel(const int *__restrict__ group_size, int64_t K,
                                                          SubTotal *__restrict__ totals)
{
    const int64_t base = (int64_t)blockIdx.x * kSubScan;
    unsigned long long m = 0, w = 0;
#pragma unroll
    for (int u = 0; u < kSubPer; ++u) {
        const int64_t k = base + u * 1024 + threadIdx.x;
        const unsigned int v = k < K ? (unsigned int)group_size[k] : 0u;
        m += v;
        w += sub_items(v);
    }
    const SubTotal t = sub_block_sum(m, w);
    if (threadIdx.x == 0) totals[blockIdx.x] = t;
}

__global__ void __launch_bounds__(1024) sub_offsets_kernel(const int *__restrict__ group_size, int64_t K,
                                                           const SubTotal *__restrict__ totals,
                                                           unsigned int *__restrict__ offsets,
                                                           unsigned int *__restrict__ cursor,
                                                           unsigned long long *__restrict__ work_off)
{
    __shared__ unsigned int s_warp[32];
    __shared__ unsigned long long s_wwarp[32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned long long pm = 0, pw = 0;
    for (unsigned int c = threadIdx.x; c < blockIdx.x; c += 1024) { pm += totals[c].members; pw += totals[c].items; }
    const SubTotal before = sub_block_sum(pm, pw);
    // warp w scans halos base + 256 w .. + 255: kSubPer coalesced rows of 32, a warp scan per row
    const int64_t k0 = (int64_t)blockIdx.x * kSubScan + (int64_t)warp * (32 * kSubPer) + lane;
    unsigned int ex[kSubPer];  // exclusive prefix inside the warp's chunk
    unsigned long long wex[kSubPer];
    unsigned int run = 0;
    unsigned long long wrun = 0;
#pragma unroll
    for (int u = 0; u < kSubPer; ++u) {
        const int64_t k = k0 + 32 * u;
        const unsigned int v = k < K ? (unsigned int)group_size[k] : 0u;
        const unsigned long long wv = sub_items(v);
        unsigned int incl = v;
        unsigned long long wincl = wv;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned int t = __shfl_up_sync(0xffffffffu, incl, o);
            const unsigned long long wt = __shfl_up_sync(0xffffffffu, wincl, o);
            if (lane >= o) { incl += t; wincl += wt; }
        }
        ex[u] = run + incl - v;
        wex[u] = wrun + wincl - wv;
        run += __shfl_sync(0xffffffffu, incl, 31);
        wrun += __shfl_sync(0xffffffffu, wincl, 31);
    }
    if (lane == 0) { s_warp[warp] = run; s_wwarp[warp] = wrun; }
    __syncthreads();
    unsigned int off = (unsigned int)before.members, tot = 0;
    unsigned long long woff = before.items, wtot = 0;
    for (int w = 0; w < 32; ++w) {
        const unsigned int t = s_warp[w];
        const unsigned long long wt = s_wwarp[w];
        if (w < warp) { off += t; woff += wt; }
        tot += t;
        wtot += wt;
    }
#pragma unroll
    for (int u = 0; u < kSubPer; ++u) {
        const int64_t k = k0 + 32 * u;
        if (k < K) { offsets[k] = off + ex[u]; cursor[k] = 0u; work_off[k] = woff + wex[u]; }
    }
    if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) {
        offsets[K] = (unsigned int)before.members + tot;
        work_off[K] = before.items + wtot;
    }
}

// members[offsets[k] + rank] = i for every particle of kept halo k; sub_labels[i] = i (R31 and the
// value every root keeps); the union-find of the slots starts as all roots.
__global__ void __launch_bounds__(kBlock) sub_fill_kernel(const int *__restrict__ particle_group, int64_t N, int64_t K,
                                                          const unsigned int *__restrict__ offsets,
                                                          unsigned int *__restrict__ cursor, int *__restrict__ members,
                                                          unsigned int *__restrict__ sub_rel,
                                                          int *__restrict__ sub_labels)
{
    const int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (i >= N) return;
    sub_labels[i] = (int)i;
    const int k = particle_group[i];
    if (k < 0 || k >= K) return;
    const unsigned int slot = offsets[k] + atomicAdd(cursor + k, 1u);
    members[slot] = (int)i;
    sub_rel[slot] = 0u;
}

// WRAP = false: the caller knows that no coordinate difference of the two tiles exceeds L / 2, where the
// minimum image is the identity.
template <bool WRAP>
__device__ __forceinline__ bool linked6(const float *a, const float *b, const Sub6 &q)
{
    float dx = __fsub_rn(a[0], b[0]), dy = __fsub_rn(a[1], b[1]), dz = __fsub_rn(a[2], b[2]);
    if (WRAP) {
        dx = min_image(dx, q.L, q.h);
        dy = min_image(dy, q.L, q.h);
        dz = min_image(dz, q.L, q.h);
    }
    const float ux = __fsub_rn(a[3], b[3]), uy = __fsub_rn(a[4], b[4]), uz = __fsub_rn(a[5], b[5]);
    const float dx2 = __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
    const float dv2 = __fadd_rn(__fadd_rn(__fmul_rn(ux, ux), __fmul_rn(uy, uy)), __fmul_rn(uz, uz));
    return __fadd_rn(__fmul_rn(dx2, q.rx), __fmul_rn(dv2, q.rv)) <= q.ell2;
}

// Bounding box of the positions of a tile (wrapped into [0, L): non-negative floats order like their bits).
struct SubBox {
    unsigned int lo[3], hi[3];
};
__device__ __forceinline__ SubBox sub_box(const float *p, bool valid)
{
    SubBox bx;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        // wrapped coordinates are >= 0, so their bit patterns order like the values -- except -0.0f (wrap1 returns it
        // unchanged), which + 0.0f turns into +0.0f
        const unsigned int bits = __float_as_uint(__fadd_rn(p[a], 0.0f));
        bx.lo[a] = __reduce_min_sync(0xffffffffu, valid ? bits : 0xffffffffu);
        bx.hi[a] = __reduce_max_sync(0xffffffffu, valid ? bits : 0u);
    }
    return bx;
}
// true if some coordinate difference between (or inside) the two boxes can exceed h = L / 2
__device__ __forceinline__ bool sub_needs_wrap(const SubBox &a, const SubBox &b, float h)
{
    bool w = false;
#pragma unroll
    for (int k = 0; k < 3; ++k)
        w = w || __fsub_rn(__uint_as_float(max(a.hi[k], b.hi[k])), __uint_as_float(min(a.lo[k], b.lo[k]))) > h;
    return w;
}

constexpr int kSubWarps = kBlock / 32;

// One warp per tile of 32 member slots; the tile meets itself and every earlier tile; a pair is
// taken by its later slot.  Two launches share the halos by size: one warp per halo of at most
// kSubSmall members (eight halos per CTA: a typical halo has two tiles); the tile rows of the larger
// halos are cut into work items of at most kSubChunk partner tiles, dealt to all warps of the grid,
// so that a halo of thousands of members is not one CTA's job (its cost is quadratic).
// Tile `it` (slots it ts .. it ts + ts - 1, ts <= 32) of the halo at member offset `off` (M members)
// against its partner tiles jt0 .. jt1 (<= it), the way link_kernel's tile role does it: the tile
// sits in registers, partner tiles are staged in shared memory as six columns, the tests of one
// candidate come out as a ballot, the tile's own components are closed in registers (rotation: lane i
// meets lane i + d, d = 1 .. 16, every unordered pair once; then breadth-first over the lanes) and
// only one hook per (component, linked candidate) reaches the union-find.  The item that holds the
// diagonal (jt1 == it) hooks and counts the tile's own pairs.
__device__ __forceinline__ void sub_tile_row(const float *__restrict__ pos, const float *__restrict__ vel,
                                             const Sub6 &q, const int *__restrict__ members,
                                             unsigned int *sub_rel, float (*s_j)[32], int off, int M, int ts, int it,
                                             int jt0, int jt1, int lane, unsigned int &nedges)
{
    constexpr unsigned int kAll = 0xffffffffu;
    const int ib = off + it * ts, myslot = ib + lane;
    const int cntI = min(ts, M - it * ts);
    const bool valid = lane < cntI;
    float me[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    int my_oi = 0x7fffffff;
    if (valid) {
        my_oi = members[myslot];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            me[a] = wrap1(__ldg(pos + 3 * (int64_t)my_oi + a), q.L);
            me[3 + a] = __ldg(vel + 3 * (int64_t)my_oi + a);
        }
    }
    // ---- the tile against itself
    __syncwarp();
#pragma unroll
    for (int a = 0; a < 6; ++a) s_j[a][lane] = me[a];
    __syncwarp();
    unsigned int adj = 0;
    const int dmax = min(16, cntI - 1);
    const SubBox boxI = sub_box(me, valid);
    if (sub_needs_wrap(boxI, boxI, q.h)) {
        for (int d = 1; d <= dmax; ++d) {
            const int c = (lane + d) & 31;
            const float pj[6] = {s_j[0][c], s_j[1][c], s_j[2][c], s_j[3][c], s_j[4][c], s_j[5][c]};
            if (valid && c < cntI && (d < 16 || lane < 16) && linked6<true>(me, pj, q)) adj |= 1u << c;
        }
    } else {
        for (int d = 1; d <= dmax; ++d) {
            const int c = (lane + d) & 31;
            const float pj[6] = {s_j[0][c], s_j[1][c], s_j[2][c], s_j[3][c], s_j[4][c], s_j[5][c]};
            if (valid && c < cntI && (d < 16 || lane < 16) && linked6<false>(me, pj, q)) adj |= 1u << c;
        }
    }
    const bool diag = jt1 == it;
    if (diag) nedges += (unsigned int)__popc(adj);
    const unsigned int self = 1u << lane;
    unsigned int grp = self;
    int head = lane;
    if (__any_sync(kAll, adj != 0u)) {
        unsigned int sym = adj;  // make it symmetric: lane k collects the lanes that found k
        for (int k = 0; k < cntI; ++k) {
            const unsigned int bal = __ballot_sync(kAll, (adj >> k) & 1u);
            if (lane == k) sym |= bal;
        }
        unsigned int todo = __ballot_sync(kAll, sym != 0u);
        while (todo) {
            const int r = __ffs((int)todo) - 1;
            unsigned int vis = 1u << r;
            while (true) {
                const unsigned int nxt = vis | __reduce_or_sync(kAll, (vis & self) ? sym : 0u);
                if (nxt == vis) break;
                vis = nxt;
            }
            const bool in = (vis & self) != 0u;
            const int m = __reduce_min_sync(kAll, in ? my_oi : 0x7fffffff);
            const unsigned int hb = __ballot_sync(kAll, in && my_oi == m);
            if (in) { grp = vis; head = __ffs((int)hb) - 1; }
            todo &= ~vis;
        }
    }
    const bool leader = head == lane;  // head: the member of my component with the smallest original index
    if (diag && !leader && atomicCAS(sub_rel + myslot, 0u, (unsigned int)(lane - head)) != 0u)
        unite_rel(sub_rel, members, myslot, ib + head);  // somebody hooked me first: general path

    // ---- the earlier tiles (all full: ts members)
    for (int jt = jt0; jt <= min(jt1, it - 1); ++jt) {
        const int jslot0 = off + jt * ts;
        __syncwarp();
        float pjl[3] = {0.f, 0.f, 0.f};
        if (lane < ts) {
            const int64_t j = members[jslot0 + lane];
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                pjl[a] = wrap1(__ldg(pos + 3 * j + a), q.L);
                s_j[a][lane] = pjl[a];
                s_j[3 + a][lane] = __ldg(vel + 3 * j + a);
            }
        }
        const bool wrap = sub_needs_wrap(boxI, sub_box(pjl, lane < ts), q.h);
        __syncwarp();
        unsigned int adjT = 0;  // lane k: tile lanes linked to candidate k
        if (wrap) {
#pragma unroll 4
            for (int k = 0; k < ts; ++k) {
                const float pj[6] = {s_j[0][k], s_j[1][k], s_j[2][k], s_j[3][k], s_j[4][k], s_j[5][k]};
                const unsigned int bal = __ballot_sync(kAll, valid && linked6<true>(me, pj, q));
                if (lane == k) adjT = bal;
            }
        } else {
#pragma unroll 4
            for (int k = 0; k < ts; ++k) {
                const float pj[6] = {s_j[0][k], s_j[1][k], s_j[2][k], s_j[3][k], s_j[4][k], s_j[5][k]};
                const unsigned int bal = __ballot_sync(kAll, valid && linked6<false>(me, pj, q));
                if (lane == k) adjT = bal;
            }
        }
        nedges += (unsigned int)__popc(adjT);
        const unsigned int active = __reduce_or_sync(kAll, adjT);
        if (!active) continue;
        unsigned int lead = __ballot_sync(kAll, leader && (grp & active));
        while (lead) {
            const int gl = __ffs((int)lead) - 1;
            lead &= lead - 1u;
            const unsigned int comp = __shfl_sync(kAll, grp, gl);
            if (adjT & comp) unite_rel(sub_rel, members, jslot0 + lane, ib + gl);  // the leader lane is the head
        }
    }
    __syncwarp();
}

// Halos of at most kSubSmall members: one warp per halo.
__global__ void __launch_bounds__(kBlock) subhalo_small_kernel(const float *__restrict__ pos,
                                                               const float *__restrict__ vel, int64_t K, Sub6 q,
                                                               const unsigned int *__restrict__ offsets,
                                                               const int *__restrict__ members, unsigned int *sub_rel,
                                                               Ctrl *ctrl)
{
    __shared__ float s_j[kSubWarps][6][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned int nedges = 0;
    for (int64_t k = (int64_t)blockIdx.x * kSubWarps + warp; k < K; k += (int64_t)gridDim.x * kSubWarps) {
        const int off = (int)offsets[k], M = (int)offsets[k + 1] - off;
        if (M > kSubSmall) continue;
        const int tiles = (M + 31) >> 5, ts = (M + tiles - 1) / max(tiles, 1);  // balanced: 41 -> 21 + 20
        for (int it = 0; it < tiles; ++it)
            sub_tile_row(pos, vel, q, members, sub_rel, s_j[warp], off, M, ts, it, 0, it, lane, nedges);
    }
    for (int o = 16; o > 0; o >>= 1) nedges += __shfl_xor_sync(0xffffffffu, nedges, o);
    if (lane == 0 && nedges) atomicAdd(&ctrl->edges, (unsigned long long)nedges);
}

// Larger halos: work item w of the whole list -> halo k (32-ary search of the item prefix `work_off`
// by the warp), then (tile row, chunk) from the triangular count of sub_items.
__global__ void __launch_bounds__(kBlock) subhalo_wide_kernel(const float *__restrict__ pos,
                                                              const float *__restrict__ vel, int64_t K, Sub6 q,
                                                              const unsigned int *__restrict__ offsets,
                                                              const unsigned long long *__restrict__ work_off,
                                                              const int *__restrict__ members, unsigned int *sub_rel,
                                                              Ctrl *ctrl)
{
    __shared__ float s_j[kSubWarps][6][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned int nedges = 0;
    const unsigned long long total = work_off[K];
    for (unsigned long long w = (unsigned long long)blockIdx.x * kSubWarps + warp; w < total;
         w += (unsigned long long)gridDim.x * kSubWarps) {
        // largest k with work_off[k] <= w (such a halo has items: work_off[k + 1] > w)
        int64_t lo = 0, hi = K;  // invariant: work_off[lo] <= w < work_off[hi]
        while (hi - lo > 1) {
            const int64_t span = hi - lo, step = (span + 31) / 32;
            const int64_t probe = lo + step * (lane + 1);
            const bool le = probe < hi && work_off[probe] <= w;
            const unsigned int bal = __ballot_sync(0xffffffffu, le);
            const int nle = __popc(bal);  // probes are increasing: the first nle of them are <= w
            const int64_t nlo = lo + step * nle, nhi = lo + step * (nle + 1);
            lo = nlo;
            hi = nhi < hi ? nhi : hi;
        }
        const int64_t k = lo;
        const int off = (int)offsets[k], M = (int)offsets[k + 1] - off;
        const unsigned long long r = w - work_off[k];
        // block row R (tile rows R kSubChunk ..): kSubChunk R (R + 1) / 2 items precede it
        long long R = (long long)((sqrt(8.0 * (double)r / kSubChunk + 1.0) - 1.0) * 0.5);
        while ((unsigned long long)kSubChunk * (unsigned long long)(R * (R + 1) / 2) > r) --R;
        while ((unsigned long long)kSubChunk * (unsigned long long)((R + 1) * (R + 2) / 2) <= r) ++R;
        const unsigned long long rem = r - (unsigned long long)kSubChunk * (unsigned long long)(R * (R + 1) / 2);
        const int it = (int)(R * kSubChunk + (long long)(rem / (unsigned long long)(R + 1)));
        const int c = (int)(rem % (unsigned long long)(R + 1));
        const int jt0 = c * kSubChunk, jt1 = min(jt0 + kSubChunk - 1, it);
        sub_tile_row(pos, vel, q, members, sub_rel, s_j[warp], off, M, 32, it, jt0, jt1, lane, nedges);
    }
    for (int o = 16; o > 0; o >>= 1) nedges += __shfl_xor_sync(0xffffffffu, nedges, o);
    if (lane == 0 && nedges) atomicAdd(&ctrl->edges, (unsigned long long)nedges);
}

// sub_labels[member] = original index of the root of its slot (roots keep their own index).
__global__ void __launch_bounds__(kBlock) sub_labels_kernel(const unsigned int *__restrict__ sub_rel,
                                                            const int *__restrict__ members,
                                                            const unsigned int *__restrict__ n_members,
                                                            int *__restrict__ sub_labels)
{
    const unsigned int total = *n_members;
    for (unsigned int s = blockIdx.x * kBlock + threadIdx.x; s < total; s += gridDim.x * kBlock) {
        int d = (int)sub_rel[s];
        if (d == 0) continue;
        int r = (int)s - d;
        while ((d = (int)sub_rel[r]) != 0) r -= d;
        sub_labels[members[s]] = members[r];
    }
}

cudaError_t launch_subgroups(const float *pos, const float *vel, const int *particle_group, const int *group_size,
                             int64_t N, int64_t K, float L, float sigma_x, float sigma_v, float ell,
                             unsigned int *offsets, unsigned int *cursor, int *members, unsigned int *sub_rel,
                             int *sub_labels, Ctrl *ctrl, int num_sms, cudaStream_t s)
{
    cudaError_t e;
    if ((e = cudaMemsetAsync(&ctrl->edges, 0, sizeof(unsigned long long), s)) != cudaSuccess) return e;
    if (N <= 0) return cudaSuccess;
    Sub6 q;
    q.L = L;
    q.h = 0.5f * L;
    q.rx = 1.0f / sigma_x;
    q.rv = 1.0f / sigma_v;
    q.ell2 = ell * ell;
    // the item prefix of the wide halos sits behind the K cursors (both inside the link's record array)
    unsigned long long *work_off = reinterpret_cast<unsigned long long *>(cursor + ((K + 2) & ~(int64_t)1));
    SubTotal *totals = reinterpret_cast<SubTotal *>(work_off + K + 1 + ((K + 1) & 1));
    const unsigned int chunks = (unsigned int)((K + kSubScan - 1) / kSubScan) + (K == 0 ? 1u : 0u);
    sub_totals_kernel<<<chunks, 1024, 0, s>>>(group_size, K, totals);
    sub_offsets_kernel<<<chunks, 1024, 0, s>>>(group_size, K, totals, offsets, cursor, work_off);
    sub_fill_kernel<<<(unsigned int)((N + kBlock - 1) / kBlock), kBlock, 0, s>>>(particle_group, N, K, offsets, cursor,
                                                                                members, sub_rel, sub_labels);
    if (K > 0) {
        const int64_t cap = (int64_t)num_sms * 16;
        const unsigned int grid_small = (unsigned int)((K + kSubWarps - 1) / kSubWarps < cap ? (K + kSubWarps - 1) / kSubWarps : cap);
        subhalo_small_kernel<<<grid_small, kBlock, 0, s>>>(pos, vel, K, q, offsets, members, sub_rel, ctrl);
        subhalo_wide_kernel<<<(unsigned int)cap, kBlock, 0, s>>>(pos, vel, K, q, offsets, work_off, members, sub_rel, ctrl);
        sub_labels_kernel<<<(unsigned int)num_sms * 8, kBlock, 0, s>>>(sub_rel, members, offsets + K, sub_labels);
    }
    return cudaGetLastError();
}

}  // namespace fof
