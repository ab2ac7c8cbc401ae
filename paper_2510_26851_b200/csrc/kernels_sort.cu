// kernels_sort.cu — H1 wrap + bin, H2 cell histogram + exclusive scan, H3 cell-contiguous reorder.
// PAPER.md:193-199 (Alg. 2: wrap, grid setup, cell indexing, sort by cell); the exclusive scan of
// the cell histogram replaces the per-particle lower/upper_bound searches of PAPER.md:203-206.
//
// Design: a two-level counting sort that never issues a global atomic per
// particle and never writes a lone 16-byte record to a random DRAM address.
//   level 1  the cell ids are cut into `bins` runs of 2^shift consecutive cells (~4096 particles
//            each).  part_hist_kernel: every CTA histograms its contiguous chunk of the input over
//            the bins in shared memory; part_offsets_kernel turns the [CTA][bin] counts into
//            write cursors (bin-major, CTA-minor exclusive scan); part_scatter_kernel re-reads the
//            chunk and writes (x, y, z, bitcast idx) records bin-contiguously.  The open write
//            streams (CTAs x bins x 32 B) fit the L2, so DRAM sees merged lines.
//   level 2  cell_sort_kernel: one CTA per bin histograms the bin's particles over its 2^shift
//            cells in shared memory, scans, writes cell_start[] coalesced, and moves every record
//            to its final place (inside the bin's window of `sorted`, L2 resident).  It also
//            initialises the union-find forest, the original-index arrays of H5 and the list of
//            dense cells of H4.
#include "fof_internal.cuh"

namespace fof {

// (wrap_cell and for_each_particle live in fof_internal.cuh: the block path uses them too)

// ---------------------------------------------------------------------------------------------
// H1 + H2 (level 1): per-CTA histogram of its chunk over the bins.
// ---------------------------------------------------------------------------------------------
template <bool VEC>
__global__ void __launch_bounds__(kPartThreads) part_hist_kernel(const float *__restrict__ pos, int64_t N, Grid g,
                                                                 int shift, int bins, int64_t chunk,
                                                                 unsigned int *__restrict__ cta_hist, Ctrl *ctrl,
                                                                 const unsigned int *gate)
{
    extern __shared__ unsigned int s_bin[];
    if (gate && *gate == 0u) return;  // the block path did the work (fof_internal.cuh Ctrl::mode)
    for (int b = threadIdx.x; b < bins; b += kPartThreads) s_bin[b] = 0u;
    __syncthreads();
    const int64_t i0 = (int64_t)blockIdx.x * chunk;
    const int64_t i1 = min(N, i0 + chunk);
    bool any_bad = false;
    for_each_particle<VEC, kPartThreads>(pos, i0, i1, [&](float x, float y, float z, int64_t) {
        const unsigned int c = wrap_cell(x, y, z, g, any_bad);
        atomicAdd(&s_bin[c >> shift], 1u);
    });
    if (any_bad) atomicOr(&ctrl->error, 1u);
    __syncthreads();
    unsigned int *dst = cta_hist + (int64_t)blockIdx.x * bins;
    for (int b = threadIdx.x; b < bins; b += kPartThreads) dst[b] = s_bin[b];
}

// ---------------------------------------------------------------------------------------------
// cta_hist[k][b] <- sum over k' < k of cta_hist[k'][b] (in place), bin_base[b] <- sum over b' < b
// of the bin totals, bin_base[bins] = N.  Block = 32 bins x 8 groups of CTAs; the last block to
// finish scans the bin totals.
// ---------------------------------------------------------------------------------------------
constexpr int kOffGroups = 8;

__global__ void __launch_bounds__(32 * kOffGroups) part_offsets_kernel(unsigned int *cta_hist, int ctas, int bins,
                                                                       unsigned int *bin_base, Ctrl *ctrl,
                                                                       const unsigned int *gate)
{
    __shared__ unsigned int s_part[kOffGroups][33];
    __shared__ unsigned int s_last;
    __shared__ unsigned int s_warp[32 * kOffGroups / 32];
    if (gate && *gate == 0u) return;  // the block path did the work (fof_internal.cuh Ctrl::mode)
    const int bx = threadIdx.x & 31, gy = threadIdx.x >> 5;
    const int b = blockIdx.x * 32 + bx;
    const int per = (ctas + kOffGroups - 1) / kOffGroups;
    const int k0 = gy * per, k1 = min(ctas, k0 + per);
    unsigned int sum = 0;
    if (b < bins)
        for (int k = k0; k < k1; ++k) sum += cta_hist[(int64_t)k * bins + b];
    s_part[gy][bx] = sum;
    __syncthreads();
    unsigned int run = 0, total = 0;
#pragma unroll
    for (int q = 0; q < kOffGroups; ++q) {
        const unsigned int t = s_part[q][bx];
        if (q < gy) run += t;
        total += t;
    }
    if (b < bins) {
        for (int k = k0; k < k1; ++k) {
            unsigned int *p = cta_hist + (int64_t)k * bins + b;
            const unsigned int t = *p;
            *p = run;
            run += t;
        }
        if (gy == 0) bin_base[b + 1] = total;  // totals, shifted by one; scanned below
    }
    // last block done: inclusive scan of bin_base[1..bins] in place, bin_base[0] = 0
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(&ctrl->scan_ticket, 1u) == gridDim.x - 1) ? 1u : 0u;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    constexpr int T = 32 * kOffGroups;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned int carry = 0;
    for (int base = 0; base < bins; base += T) {
        const int j = base + threadIdx.x;
        const unsigned int v = (j < bins) ? ((volatile unsigned int *)bin_base)[j + 1] : 0u;
        unsigned int incl = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        unsigned int off = carry, tot = 0;
#pragma unroll
        for (int w = 0; w < T / 32; ++w) {
            const unsigned int t = s_warp[w];
            if (w < warp) off += t;
            tot += t;
        }
        if (j < bins) bin_base[j + 1] = off + incl;
        carry += tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) bin_base[0] = 0u;
}

// ---------------------------------------------------------------------------------------------
// H3 (level 1): bin-contiguous records.  Same chunk -> CTA map as part_hist_kernel, so the
// shared-memory cursors (cta_hist + bin_base) hand out exactly the slots that were counted.
// ---------------------------------------------------------------------------------------------
template <bool VEC>
__global__ void __launch_bounds__(kPartThreads) part_scatter_kernel(const float *__restrict__ pos, int64_t N, Grid g,
                                                                    int shift, int bins, int64_t chunk,
                                                                    const unsigned int *__restrict__ cta_hist,
                                                                    const unsigned int *__restrict__ bin_base,
                                                                    float4 *__restrict__ part, int *__restrict__ labels,
                                                                    bool labels_vec, const unsigned int *gate,
                                                                    int *__restrict__ cnt)
{
    extern __shared__ unsigned int s_bin[];
    if (gate && *gate == 0u) return;  // the block path did the work (fof_internal.cuh Ctrl::mode)
    const unsigned int *src = cta_hist + (int64_t)blockIdx.x * bins;
    for (int b = threadIdx.x; b < bins; b += kPartThreads) s_bin[b] = src[b] + bin_base[b];
    __syncthreads();
    const int64_t i0 = (int64_t)blockIdx.x * chunk;
    const int64_t i1 = min(N, i0 + chunk);
    bool bad = false;
    for_each_particle<VEC, kPartThreads>(pos, i0, i1, [&](float x, float y, float z, int64_t i) {
        const unsigned int c = wrap_cell(x, y, z, g, bad);
        const unsigned int dst = atomicAdd(&s_bin[c >> shift], 1u);
        part[dst] = make_float4(x, y, z, __int_as_float((int)i));
    });
    // H5, first half: labels[i] = i, coalesced, while this CTA walks its chunk in the original order.
    // That is already the final label of every root (singletons above all); write_labels_kernel then
    // scatters only the labels of non-roots.
    for (int64_t i = i0 + 4 * (int64_t)threadIdx.x; i < i1; i += 4 * (int64_t)kPartThreads) {
        if (labels_vec && i + 4 <= i1) {
            *reinterpret_cast<int4 *>(labels + i) = make_int4((int)i, (int)i + 1, (int)i + 2, (int)i + 3);
        } else {
            for (int k = 0; k < 4 && i + k < i1; ++k) labels[i + k] = (int)(i + k);
        }
        // the size counters of H6 (write_labels_kernel adds to them) start at 0; cnt is a workspace array: aligned
        if (i + 4 <= i1) *reinterpret_cast<int4 *>(cnt + i) = make_int4(0, 0, 0, 0);
        else
            for (int k = 0; k < 4 && i + k < i1; ++k) cnt[i + k] = 0;
    }
}

// ---------------------------------------------------------------------------------------------
// H2 + H3 (level 2): one CTA per bin.  Shared memory: one counter per cell of the bin.
//   1. histogram of the bin's records over its cells (shared-memory atomics);
//   2. exclusive scan -> cell_start[] (coalesced), work items of the tile role of link_kernel (dense cells);
//   3. records re-read (L2) and moved to their final slot; rel = 0 (every particle a root),
//      idx_s = original index (the order of the union-find, input of H5).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned int cell_of(const float4 &v, const Grid &g)
{
    return cell_id(cell1(v.x, g), cell1(v.y, g), cell1(v.z, g), g.n);
}

__global__ void __launch_bounds__(kCellSortThreads) cell_sort_kernel(
    const float4 *__restrict__ part, const unsigned int *__restrict__ bin_base, Grid g, int shift, int64_t C,
    unsigned int *__restrict__ cell_start, float4 *sorted, unsigned int *__restrict__ rel,
    int *__restrict__ idx_s, unsigned long long *__restrict__ dense_list, Ctrl *ctrl, const unsigned int *gate)
{
    extern __shared__ unsigned int s_cell[];  // [2^shift]
    __shared__ unsigned long long s_warp[kCellSortThreads / 32];
    __shared__ unsigned int s_dbase;
    if (gate && *gate == 0u) return;  // the block path did the work (fof_internal.cuh Ctrl::mode)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int cpb = 1 << shift;
    const int64_t cell0 = (int64_t)blockIdx.x << shift;
    const int ncell = (int)min((int64_t)cpb, C - cell0);
    const unsigned int p0 = bin_base[blockIdx.x], p1 = bin_base[blockIdx.x + 1];

    for (int c = tid; c < cpb; c += kCellSortThreads) s_cell[c] = 0u;
    __syncthreads();
    // four records in flight per thread
    for (unsigned int p = p0 + tid; p < p1; p += 4 * kCellSortThreads) {
        float4 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) v[u] = __ldg(part + min(p + u * kCellSortThreads, p1 - 1));
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (p + u * kCellSortThreads < p1) atomicAdd(&s_cell[cell_of(v[u], g) - (unsigned int)cell0], 1u);
    }
    __syncthreads();

    // thread t owns cells [t * per, (t + 1) * per); (count, dense cells) packed in one 64-bit scan
    const int per = cpb / kCellSortThreads;  // 8 .. 64, multiple of 4
    const int c_lo = tid * per;
    unsigned long long mine = 0;
    for (int k = 0; k < per; k += 4) {
        const uint4 v = *reinterpret_cast<const uint4 *>(s_cell + c_lo + k);
        const unsigned int a[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            mine += a[u];
            if (a[u] >= (unsigned int)kDenseCell) mine += (unsigned long long)(dense_tiles(a[u]) * dense_parts(a[u])) << 32;
        }
    }
    unsigned long long incl = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    unsigned long long woff = 0, total = 0;
#pragma unroll
    for (int w = 0; w < kCellSortThreads / 32; ++w) {
        const unsigned long long t = s_warp[w];
        if (w < warp) woff += t;
        total += t;
    }
    if (tid == 0) {
        const unsigned int nd = (unsigned int)(total >> 32);
        s_dbase = nd ? atomicAdd(&ctrl->ndense, nd) : 0u;
    }
    __syncthreads();
    const unsigned long long excl = woff + incl - mine;
    unsigned int run = p0 + (unsigned int)excl;
    unsigned int drun = s_dbase + (unsigned int)(excl >> 32);
    for (int k = 0; k < per; k += 4) {
        uint4 v = *reinterpret_cast<const uint4 *>(s_cell + c_lo + k);
        unsigned int a[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const unsigned int cnt = a[u];
            a[u] = run;
            if (cnt >= (unsigned int)kDenseCell) {
                // one work item per (dense cell, tile of <= 32 particles, part of the tile's candidate stream)
                const unsigned int nt = dense_tiles(cnt), ts = dense_tile_size(cnt), np = dense_parts(cnt);
                for (unsigned int t = 0; t < nt; ++t)
                    for (unsigned int part = 0; part < np; ++part)
                        dense_list[drun++] = ((unsigned long long)(cell0 + c_lo + k + u) << 32) | (part << 29) |
                                             (t << 5) | (ts - 1u);
            }
            run += cnt;
        }
        v = make_uint4(a[0], a[1], a[2], a[3]);
        *reinterpret_cast<uint4 *>(s_cell + c_lo + k) = v;  // now the write cursor of each cell
        if (c_lo + k + 3 < ncell) *reinterpret_cast<uint4 *>(cell_start + cell0 + c_lo + k) = v;
        else {
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (c_lo + k + u < ncell) cell_start[cell0 + c_lo + k + u] = a[u];
        }
    }
    if (cell0 + ncell == C && tid == 0) cell_start[C] = p1;
    __syncthreads();

    for (unsigned int p = p0 + tid; p < p1; p += 4 * kCellSortThreads) {
        float4 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) v[u] = __ldg(part + min(p + u * kCellSortThreads, p1 - 1));
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (p + u * kCellSortThreads < p1)
                sorted[atomicAdd(&s_cell[cell_of(v[u], g) - (unsigned int)cell0], 1u)] = v[u];
    }
    __syncthreads();
    // the per-particle arrays of H4 / H5, written coalesced from the records this CTA just placed
    for (unsigned int p = p0 + tid; p < p1; p += kCellSortThreads) {
        const int oi = __float_as_int(__ldcg(&sorted[p].w));
        rel[p] = 0u;
        idx_s[p] = oi;
    }
}

// ---------------------------------------------------------------------------------------------
// Second partition pass (only when there are more than kTwoPassBins bins): the input is the
// coarse-bin-contiguous record array of a first pass over bins 2^kCoarseShift times wider (a few
// dozen write streams per CTA, each a long run), so a CTA's contiguous chunk only touches ~1000 fine
// bins inside one coarse bin (tens of MB): the open write streams stay in the L2 and in the TLB.  At
// 512^3 a single pass has 148 CTAs x 32768 streams spread over 2 GB: 4.7 ms; two passes: 3.3 ms
// (measured with 2^6 .. 2^11: 5.0, 5.2 (2^8), 3.6, 3.3, 3.8 ms).
// ---------------------------------------------------------------------------------------------
#ifndef FOF_TWO_PASS_BINS
#define FOF_TWO_PASS_BINS 8192
#endif
constexpr int kTwoPassBins = FOF_TWO_PASS_BINS;
#ifndef FOF_COARSE_SHIFT
#define FOF_COARSE_SHIFT 10
#endif
constexpr int kCoarseShift = FOF_COARSE_SHIFT;

__global__ void __launch_bounds__(kPartThreads) rec_hist_kernel(const float4 *__restrict__ rec, int64_t N, Grid g,
                                                                int shift, int bins, int64_t chunk,
                                                                unsigned int *__restrict__ cta_hist,
                                                                const unsigned int *gate)
{
    extern __shared__ unsigned int s_bin[];
    if (gate && *gate == 0u) return;  // the block path did the work (fof_internal.cuh Ctrl::mode)
    for (int b = threadIdx.x; b < bins; b += kPartThreads) s_bin[b] = 0u;
    __syncthreads();
    const int64_t i0 = (int64_t)blockIdx.x * chunk, i1 = min(N, i0 + chunk);
    for (int64_t i = i0 + threadIdx.x; i < i1; i += 4 * kPartThreads) {
        float4 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) v[u] = __ldg(rec + min(i + u * kPartThreads, i1 - 1));
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (i + u * kPartThreads < i1) atomicAdd(&s_bin[cell_of(v[u], g) >> shift], 1u);
    }
    __syncthreads();
    unsigned int *dst = cta_hist + (int64_t)blockIdx.x * bins;
    for (int b = threadIdx.x; b < bins; b += kPartThreads) dst[b] = s_bin[b];
}

__global__ void __launch_bounds__(kPartThreads) rec_scatter_kernel(const float4 *__restrict__ rec, int64_t N, Grid g,
                                                                   int shift, int bins, int64_t chunk,
                                                                   const unsigned int *__restrict__ cta_hist,
                                                                   const unsigned int *__restrict__ bin_base,
                                                                   float4 *__restrict__ out, const unsigned int *gate)
{
    extern __shared__ unsigned int s_bin[];
    if (gate && *gate == 0u) return;  // the block path did the work (fof_internal.cuh Ctrl::mode)
    const unsigned int *src = cta_hist + (int64_t)blockIdx.x * bins;
    for (int b = threadIdx.x; b < bins; b += kPartThreads) s_bin[b] = src[b] + bin_base[b];
    __syncthreads();
    const int64_t i0 = (int64_t)blockIdx.x * chunk, i1 = min(N, i0 + chunk);
    for (int64_t i = i0 + threadIdx.x; i < i1; i += 4 * kPartThreads) {
        float4 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) v[u] = __ldg(rec + min(i + u * kPartThreads, i1 - 1));
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (i + u * kPartThreads < i1) out[atomicAdd(&s_bin[cell_of(v[u], g) >> shift], 1u)] = v[u];
    }
}

static inline cudaError_t set_smem(const void *fn, size_t bytes)
{
    if (bytes <= 40 * 1024) return cudaSuccess;  // static shared memory counts against the 48 KB default too
    return cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

cudaError_t launch_sort(const float *pos, int64_t N, Grid g, const SortPlan &sp, int ctas, unsigned int *cta_hist,
                        unsigned int *bin_base, float4 *part, unsigned int *cell_start, float4 *sorted,
                        unsigned int *rel, int *idx_s, unsigned long long *dense_list, int *labels, Ctrl *ctrl,
                        const unsigned int *gate, int *cnt, StageHook &hook, cudaStream_t s)
{
    if (N <= 0) return cudaSuccess;
    const size_t smem_bins = (size_t)sp.bins * sizeof(unsigned int);
    const size_t smem_cells = ((size_t)1 << sp.shift) * sizeof(unsigned int);
    cudaError_t e;
    const bool vec = ((uintptr_t)pos & 15) == 0;
    auto hist = vec ? part_hist_kernel<true> : part_hist_kernel<false>;
    auto scat = vec ? part_scatter_kernel<true> : part_scatter_kernel<false>;
    if ((e = set_smem((const void *)hist, smem_bins)) != cudaSuccess) return e;
    if ((e = set_smem((const void *)scat, smem_bins)) != cudaSuccess) return e;
    if ((e = set_smem((const void *)cell_sort_kernel, smem_cells)) != cudaSuccess) return e;
    const int64_t chunk = ((N + ctas - 1) / ctas + 3) & ~(int64_t)3;  // a multiple of 4: quads stay aligned
    const int64_t C = (int64_t)g.n * g.n * g.n;
    const bool labels_vec = ((uintptr_t)labels & 15) == 0;
    if (sp.bins <= kTwoPassBins) {
        hook.begin(0, 1);
        hist<<<ctas, kPartThreads, smem_bins, s>>>(pos, N, g, sp.shift, sp.bins, chunk, cta_hist, ctrl, gate);
        hook.end(0);
        hook.begin(1, 1);
        part_offsets_kernel<<<(sp.bins + 31) / 32, 32 * kOffGroups, 0, s>>>(cta_hist, ctas, sp.bins, bin_base, ctrl, gate);
        hook.end(1);
        hook.begin(2, 1);
        scat<<<ctas, kPartThreads, smem_bins, s>>>(pos, N, g, sp.shift, sp.bins, chunk, cta_hist, bin_base, part, labels,
                                                   labels_vec, gate, cnt);
        hook.end(2);
    } else {
        // pass 1 over bins 2^kCoarseShift times wider: pos -> `sorted` (used as scratch); pass 2: -> `part`
        const int cshift = sp.shift + kCoarseShift;
        const int cbins = (int)((C + ((int64_t)1 << cshift) - 1) >> cshift);
        unsigned int *cbase = bin_base + sp.bins + 2;  // the coarse bin offsets live behind the fine ones
        if ((e = set_smem((const void *)rec_hist_kernel, smem_bins)) != cudaSuccess) return e;
        if ((e = set_smem((const void *)rec_scatter_kernel, smem_bins)) != cudaSuccess) return e;
        const size_t smem_c = (size_t)cbins * sizeof(unsigned int);
        hook.begin(0, 1);
        hist<<<ctas, kPartThreads, smem_c, s>>>(pos, N, g, cshift, cbins, chunk, cta_hist, ctrl, gate);
        hook.end(0);
        hook.begin(1, 2);
        part_offsets_kernel<<<(cbins + 31) / 32, 32 * kOffGroups, 0, s>>>(cta_hist, ctas, cbins, cbase, ctrl, gate);
        hook.end(1);
        hook.begin(2, 3);
        scat<<<ctas, kPartThreads, smem_c, s>>>(pos, N, g, cshift, cbins, chunk, cta_hist, cbase, sorted, labels,
                                                labels_vec, gate, cnt);
        rec_hist_kernel<<<ctas, kPartThreads, smem_bins, s>>>(sorted, N, g, sp.shift, sp.bins, chunk, cta_hist, gate);
        if ((e = cudaMemsetAsync(&ctrl->scan_ticket, 0, sizeof(unsigned int), s)) != cudaSuccess) return e;
        part_offsets_kernel<<<(sp.bins + 31) / 32, 32 * kOffGroups, 0, s>>>(cta_hist, ctas, sp.bins, bin_base, ctrl, gate);
        rec_scatter_kernel<<<ctas, kPartThreads, smem_bins, s>>>(sorted, N, g, sp.shift, sp.bins, chunk, cta_hist,
                                                                 bin_base, part, gate);
        hook.end(2);
    }
    hook.begin(3, 1);
    cell_sort_kernel<<<sp.bins, kCellSortThreads, smem_cells, s>>>(part, bin_base, g, sp.shift, C, cell_start, sorted,
                                                                  rel, idx_s, dense_list, ctrl, gate);
    hook.end(3);
    return cudaGetLastError();
}

}  // namespace fof
