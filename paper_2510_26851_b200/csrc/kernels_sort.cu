// kernels_sort.cu — H1 wrap + bin, H2 cell histogram + exclusive scan, H3 cell-contiguous reorder.
// PAPER.md:193-199 (Alg. 2: wrap, grid setup, cell indexing, sort by cell); the exclusive scan of
// the cell histogram replaces the per-particle lower/upper_bound searches of PAPER.md:203-206.
#include "fof_internal.cuh"

namespace fof {

// ---------------------------------------------------------------------------------------------
// H1 + first half of H2: one thread per particle.  Reads pos once; the atomicAdd on the cell
// counter returns the particle's rank inside its cell, which makes H3 atomic-free.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kBlock) bin_kernel(const float *__restrict__ pos, int64_t N, Grid g,
                                                     unsigned int *__restrict__ cell_count,
                                                     unsigned int *__restrict__ rank, Ctrl *ctrl)
{
    int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (i >= N) return;
    float x = pos[3 * i + 0], y = pos[3 * i + 1], z = pos[3 * i + 2];
    if (!(isfinite(x) && isfinite(y) && isfinite(z))) {
        atomicOr(&ctrl->error, 1u);
        x = y = z = 0.0f;
    }
    x = wrap1(x, g.L);
    y = wrap1(y, g.L);
    z = wrap1(z, g.L);
    unsigned int c = cell_id(cell1(x, g), cell1(y, g), cell1(z, g), g.n);
    rank[i] = atomicAdd(cell_count + c, 1u);
}

// ---------------------------------------------------------------------------------------------
// H2: single-pass exclusive scan (decoupled look-back) over the cell counters, in place.
// state[tile] = (flag << 32) | value, flag 1 = tile aggregate, 2 = inclusive prefix; one 64-bit
// word so that flag and value are published together.  Tiles are handed out by an atomic ticket,
// so a tile only ever waits on tiles that already started.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned int lookback(unsigned long long *state, unsigned int tile, unsigned int aggregate,
                                                 int lane)
{
    // executed by one full warp; returns the exclusive prefix of `tile` (valid in every lane)
    unsigned int exclusive = 0;
    int64_t idx = (int64_t)tile - 1;
    while (true) {
        int64_t j = idx - lane;
        unsigned long long v = (2ull << 32);  // tiles before 0: prefix 0
        if (j >= 0) {
            do { v = ld_relaxed_u64(state + j); } while ((v >> 32) == 0);
        }
        unsigned int flag = (unsigned int)(v >> 32), val = (unsigned int)v;
        unsigned int full = __ballot_sync(0xffffffffu, flag == 2);
        int stop = full ? __ffs(full) - 1 : 31;           // nearest predecessor with a full prefix
        unsigned int part = (lane <= stop) ? val : 0;
        for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
        exclusive += part;
        if (full) break;
        idx -= 32;
    }
    if (lane == 0) st_relaxed_u64(state + tile, (2ull << 32) | (unsigned long long)(exclusive + aggregate));
    return exclusive;
}

__global__ void __launch_bounds__(kBlock) cell_scan_kernel(unsigned int *data, int64_t n_items,
                                                           unsigned long long *state, Ctrl *ctrl,
                                                           unsigned int *__restrict__ dense_list)
{
    __shared__ unsigned int s_tile, s_prefix;
    __shared__ unsigned int s_warp[kBlock / 32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(&ctrl->scan_ticket, 1u);
    __syncthreads();
    const unsigned int tile = s_tile;
    const int64_t base = (int64_t)tile * kScanTile + (int64_t)tid * kScanItems;

    unsigned int v[kScanItems];
    if (base + kScanItems <= n_items) {
        const uint4 a = *reinterpret_cast<const uint4 *>(data + base);
        const uint4 b = *reinterpret_cast<const uint4 *>(data + base + 4);
        v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
    } else {
#pragma unroll
        for (int k = 0; k < kScanItems; ++k) v[k] = (base + k < n_items) ? data[base + k] : 0u;
    }
    // cells holding kDenseCell..kDenseMax particles are listed for link_dense_kernel (order is
    // irrelevant); one atomic per warp that has any
    {
        unsigned int nd = 0;
#pragma unroll
        for (int k = 0; k < kScanItems; ++k)
            nd += (v[k] >= (unsigned int)kDenseCell && v[k] <= (unsigned int)kDenseMax) ? 1u : 0u;
        if (__any_sync(0xffffffffu, nd != 0u)) {
            unsigned int incl_d = nd;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const unsigned int t = __shfl_up_sync(0xffffffffu, incl_d, o);
                if (lane >= o) incl_d += t;
            }
            unsigned int wbase = 0;
            if (lane == 31) wbase = atomicAdd(&ctrl->ndense, incl_d);
            wbase = __shfl_sync(0xffffffffu, wbase, 31);
            unsigned int dst = wbase + incl_d - nd;
#pragma unroll
            for (int k = 0; k < kScanItems; ++k)
                if (v[k] >= (unsigned int)kDenseCell && v[k] <= (unsigned int)kDenseMax)
                    dense_list[dst++] = (unsigned int)(base + k);
        }
    }
    unsigned int sum = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) { unsigned int t = v[k]; v[k] = sum; sum += t; }  // thread-exclusive
    unsigned int incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        unsigned int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    unsigned int warp_off = 0, total = 0;
#pragma unroll
    for (int w = 0; w < kBlock / 32; ++w) {
        unsigned int t = s_warp[w];
        if (w < warp) warp_off += t;
        total += t;
    }
    if (warp == 0) {
        if (tile == 0) {
            if (lane == 0) { st_relaxed_u64(state, (2ull << 32) | total); s_prefix = 0; }
        } else {
            if (lane == 0) st_relaxed_u64(state + tile, (1ull << 32) | total);
            unsigned int ex = lookback(state, tile, total, lane);
            if (lane == 0) s_prefix = ex;
        }
    }
    __syncthreads();
    const unsigned int off = s_prefix + warp_off + (incl - sum);
    if (base + kScanItems <= n_items) {
        uint4 a = make_uint4(v[0] + off, v[1] + off, v[2] + off, v[3] + off);
        uint4 b = make_uint4(v[4] + off, v[5] + off, v[6] + off, v[7] + off);
        *reinterpret_cast<uint4 *>(data + base) = a;
        *reinterpret_cast<uint4 *>(data + base + 4) = b;
    } else {
#pragma unroll
        for (int k = 0; k < kScanItems; ++k)
            if (base + k < n_items) data[base + k] = v[k] + off;
    }
}

// ---------------------------------------------------------------------------------------------
// H3: reorder particles cell-contiguously; sorted[j] = (wx, wy, wz, bitcast(original index)).
// dst = cell_start[cell] + rank: no atomics, the cell id is recomputed from pos (bit-identical
// to H1 because it is the same code on the same input).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kBlock) scatter_kernel(const float *__restrict__ pos, int64_t N, Grid g,
                                                         const unsigned int *__restrict__ cell_start,
                                                         const unsigned int *__restrict__ rank,
                                                         float4 *__restrict__ sorted)
{
    int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (i >= N) return;
    float x = pos[3 * i + 0], y = pos[3 * i + 1], z = pos[3 * i + 2];
    if (!(isfinite(x) && isfinite(y) && isfinite(z))) x = y = z = 0.0f;
    x = wrap1(x, g.L);
    y = wrap1(y, g.L);
    z = wrap1(z, g.L);
    unsigned int c = cell_id(cell1(x, g), cell1(y, g), cell1(z, g), g.n);
    unsigned int dst = cell_start[c] + rank[i];
    sorted[dst] = make_float4(x, y, z, __int_as_float((int)i));
}

static inline unsigned int blocks_for(int64_t n, int per_block) { return (unsigned int)((n + per_block - 1) / per_block); }

cudaError_t launch_bin(const float *pos, int64_t N, Grid g, unsigned int *cell_count, unsigned int *rank,
                       Ctrl *ctrl, cudaStream_t s)
{
    if (N > 0) bin_kernel<<<blocks_for(N, kBlock), kBlock, 0, s>>>(pos, N, g, cell_count, rank, ctrl);
    return cudaGetLastError();
}

cudaError_t launch_cell_scan(unsigned int *cell, int64_t n_items, unsigned long long *state, Ctrl *ctrl,
                             unsigned int *dense_list, int64_t tiles, cudaStream_t s)
{
    cell_scan_kernel<<<(unsigned int)tiles, kBlock, 0, s>>>(cell, n_items, state, ctrl, dense_list);
    return cudaGetLastError();
}

cudaError_t launch_scatter(const float *pos, int64_t N, Grid g, const unsigned int *cell_start,
                           const unsigned int *rank, float4 *sorted, cudaStream_t s)
{
    if (N > 0) scatter_kernel<<<blocks_for(N, kBlock), kBlock, 0, s>>>(pos, N, g, cell_start, rank, sorted);
    return cudaGetLastError();
}

}  // namespace fof
