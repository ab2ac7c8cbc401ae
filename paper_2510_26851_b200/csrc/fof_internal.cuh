// fof_internal.cuh — plan, workspace layout and the device-side arithmetic shared by the kernels
// of libfof_b200.so.  sm_100a only.  Nothing here is shared with oracle/ (the CPU oracle is an
// independent restatement of the paper).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/fof.h"

namespace fof {

constexpr int kBlock = 256;           // threads per CTA for the streaming kernels
#ifndef FOF_SCAN_ITEMS
#define FOF_SCAN_ITEMS 32
#endif
constexpr int kScanItems = FOF_SCAN_ITEMS;  // items per thread in the single-pass scan (multiple of 4)
constexpr int kScanTile = kBlock * kScanItems;
constexpr float kCellMargin = 1.001f; // cell side >= b * kCellMargin  (R3)
constexpr int kMaxGrid = 1024;        // n^3 <= 2^30: at most kMaxBins bins of 2^15 cells
constexpr int kPartThreads = 1024;    // threads per CTA of the level-1 partition kernels
constexpr int kCellSortThreads = 512; // threads per CTA of the level-2 cell sort
constexpr int kMinShift = 12;         // a bin is 2^shift consecutive cell ids, shift in [12, 15]
constexpr int kMaxBins = 32768;       // level-1 bins (one shared-memory counter each)
constexpr int kMaxPartCtas = 512;     // CTAs of the level-1 kernels (one per SM)
constexpr int kMaxStages = 24;        // profiled stages (fof_profile_*)

// Device control block at the start of the workspace (zeroed at the start of fof_link).
struct Ctrl {
    unsigned int error;        // bit 0: non-finite position seen
    unsigned int scan_ticket;  // blocks of part_offsets_kernel that have finished
    unsigned int gscan_ticket; // dynamic tile id for the group compaction scan
    unsigned int pad0;
    unsigned long long edges;       // true edges (unordered pairs with d2 <= b2)
    unsigned long long pair_tests;  // distance tests executed
    long long K;                    // kept groups (written by fof_groups)
    unsigned long long grid_pairs;  // candidate pairs of the unfiltered half stencil on this grid
    unsigned int ndense;            // work items (dense cell, tile) listed by cell_sort_kernel
    unsigned int tile_ticket;       // next (dense cell, tile) item of link_kernel
    unsigned int sparse_ticket;     // next 32-particle chunk of link_kernel
    unsigned int mode;              // block path: 0 = every block fits shared memory, 1 = fall back to the cell path
    unsigned int ncross;            // block path: equivalence pairs listed by block_link_kernel
    unsigned int tile_ticket2;      // block path: next input tile of block_scatter_kernel
    unsigned int max_block;         // block path: records (own + ghost) of the fullest block
    unsigned int pad1[3];
    unsigned long long edges_b;      // block path: true edges / distance tests of block_link_kernel (kept apart from the
    unsigned long long pair_tests_b; // cell path's: after a late fall-back both kernels have counted)
};
static_assert(sizeof(Ctrl) <= 256, "Ctrl must fit its 256-byte slot");

// Everything a kernel needs to know about the box and the grid, passed by value.
struct Grid {
    float L;        // box side
    float h;        // 0.5 * L
    float b2;       // fl(b * b)
    float inv_cell; // fl(n / L)
    int n;          // cells per axis
    int n_minus_1;
    float reach;    // b in cell units + slack: how close to a cell face a particle must be to have
                    // a partner in the cell behind it (kernels_link.cu candidate_ranges)
};

// Block path (kernels_block.cu): the cell grid is cut into blocks of 2^sx x 2^sy x 2^sz cells; one CTA links
// one block out of shared memory.  Local cell grid of a block: X x Y x Z cells = its own cells plus one
// ghost layer on both x and y sides and on the upper z side (the forward half stencil never looks down in z).
struct BlockGeom {
    int sx, sy, sz;     // log2 of the block's cells per axis
    int nbx, nby, nbz;  // blocks per axis = ceil(n / 2^s); >= 3 each
    int bins;           // nbx * nby * nbz
    int X, Y, Z;        // local grid: 2^sx + 2, 2^sy + 2, 2^sz + 1
    int ncell;          // X * Y * Z
};
#ifndef FOF_BLOCK_THREADS
#define FOF_BLOCK_THREADS 512
#endif
#ifndef FOF_BLOCK_CAP
#define FOF_BLOCK_CAP 4096
#endif
constexpr int kBlockCap = FOF_BLOCK_CAP;      // most records (own + ghost) of a block that block_link_kernel holds
constexpr int kBlockThreads = FOF_BLOCK_THREADS;   // threads per CTA of block_link_kernel
constexpr int kMaxBlockBins = 16384; // most blocks (one shared-memory counter each in the partition)
constexpr unsigned int kGhostBit = 0x80000000u;  // record.w = original index | kGhostBit for a ghost copy

constexpr int kLinkBlock = 256;     // threads per CTA of the link kernels
#ifndef FOF_DENSE_CELL
#define FOF_DENSE_CELL 8
#endif
constexpr int kDenseCell = FOF_DENSE_CELL;  // cells with >= kDenseCell particles are DENSE: the pairs whose home cell is
                                            // dense belong to the tile role of link_kernel, all others to its sparse role

// A dense cell of m particles is cut into dense_tiles(m) tiles of dense_tile_size(m) <= 32
// consecutive particles (balanced: 43 -> 22 + 21, not 32 + 11); one work item per tile.
__host__ __device__ __forceinline__ unsigned int dense_tiles(unsigned int m) { return (m + 31u) >> 5; }
__host__ __device__ __forceinline__ unsigned int dense_tile_size(unsigned int m)
{
    const unsigned int T = dense_tiles(m);
    return T <= 16u ? (m + T - 1u) / T : 32u;
}
// A tile of a HEAVY cell (>= kHeavyCell particles: a clump core) meets thousands of candidates; its
// candidate stream (earlier tiles of the cell + 13 forward cells) is dealt round-robin to
// dense_parts(m) work items so that no single warp carries it (the tail of the link kernel).
#ifndef FOF_HEAVY_CELL
#define FOF_HEAVY_CELL 128
#endif
#ifndef FOF_HEAVY_PARTS
#define FOF_HEAVY_PARTS 8
#endif
constexpr unsigned int kHeavyCell = FOF_HEAVY_CELL, kHeavyParts = FOF_HEAVY_PARTS;  // parts: a power of two <= 8
__host__ __device__ __forceinline__ unsigned int dense_parts(unsigned int m)
{
    return (m >= kHeavyCell && m < (1u << 29)) ? kHeavyParts : 1u;  // item word: part:3 | tile:24 | size:5
}



}  // namespace fof

namespace fof {
struct SortPlan {
    int shift;  // cells per bin = 2^shift
    int bins;   // ceil(C / 2^shift) <= kMaxBins
};


}  // namespace fof

struct fof_handle {
    int64_t N;
    float L, b;
    int32_t N_min;
    int32_t n, n_max;
    int64_t C;  // n^3
    fof::Grid grid;
    // workspace layout (byte offsets, 256-B aligned)
    fof::SortPlan sort;
    fof::BlockGeom bg;      // block path geometry (valid if block_ok)
    bool block_ok;          // the plan admits the block path (>= 3 blocks per axis, <= kMaxBlockBins blocks)
    int path;               // FOF_PATH_AUTO / FOF_PATH_BLOCKS / FOF_PATH_CELLS
    size_t off_cursor;      // block path: records written to every block's slice so far
    size_t off_ctrl, off_cell, off_part, off_cta_hist, off_bin_base, off_sorted, off_cnt, off_acc, off_gscan_state;
    size_t off_rel, off_idx, off_dense;  // union-find (cell-sorted space), original index of each slot, work items
    size_t ws_bytes;
    int64_t gscan_tiles, max_groups;
    int num_sms, part_ctas;
    bool linked;
    bool counted;           // the last fof_link left the group sizes of `counted_labels` in the workspace (H6 done)
    const void *counted_labels;
    bool linked_cells;      // the last fof_link left cell_start / sorted / idx_s / rel in the workspace for certain
    const void *linked_ws;
    char cuda_err[256];
    // measurement aids
    int prof_slots;        // 0 = profiling off; else event sets used round-robin, one per fof_link call
    int prof_only;         // -1: every stage is timed; k: only stage k (fof_profile_only)
    int prof_cur;          // slot of the current (last) fof_link
    cudaEvent_t *ev;       // [slot][2k] before, [slot][2k+1] after stage k
    bool *ev_valid;        // [slot][k]
    unsigned long long launches;
    // fof_run_host: the labels go back to the host on a stream of their own while the groups are built
    cudaStream_t copy_stream;
    cudaEvent_t ev_linked;
    // fof_host_submit / fof_host_wait: two inputs in flight, host -> device, compute and device -> host streams
    struct HostSlot {
        bool busy;
        cudaStream_t out;            // this slot's device -> host copies
        cudaEvent_t ev_in, ev_linked, ev_groups, ev_ctrl;
        fof::Ctrl *ctrl_pin;         // pinned copy of the workspace's Ctrl (K, error bits) taken after the groups
        int64_t cap;
        int32_t *group_label_host, *group_size_host;
        float *group_mass_host, *group_com_host;
        const int *glabel, *gsize;   // device side of the group records (in the slot's dev_buf)
        const float *gmass, *gcom;
    } slot[2];
    cudaStream_t in_stream, run_stream;
    // the potential-edge list the last fof_stochastic_list_build on this handle filled (nullptr: none is valid)
    const void *slist;
    float slist_b_link, slist_alpha;
    const void *slist_counts_ws;  // the workspace whose group-size counters hold the record counts of the current link
};

namespace fof {

// ---- wrap into [0, L): "X <- X mod L" (R6).  Explicit _rn intrinsics so
// that nvcc cannot contract the multiply-subtract into an FMA.
__device__ __forceinline__ float wrap1(float x, float L)
{
    if (x >= 0.0f && x < L) return x;
    float t = __fdiv_rn(x, L);
    float w = __fsub_rn(x, __fmul_rn(L, floorf(t)));
    if (w < 0.0f) w = __fadd_rn(w, L);
    if (!(w >= 0.0f) || w >= L) w = 0.0f;  // |x| beyond ~2^24 L: x - L floor(x / L) is off by whole ulps of x (R6)
    return w;
}

// ---- cell coordinate of a wrapped coordinate ("cell triple"); monotone in w.
__device__ __forceinline__ int cell1(float w, const Grid &g)
{
    int c = __float2int_rd(__fmul_rn(w, g.inv_cell));
    return min(max(c, 0), g.n_minus_1);
}

// linear id, x fastest (c = i_x + n_x (i_y + n_y i_z))
__device__ __forceinline__ unsigned int cell_id(int cx, int cy, int cz, int n)
{
    return (unsigned int)cx + (unsigned int)n * ((unsigned int)cy + (unsigned int)n * (unsigned int)cz);
}

// wrapped position (non-finite -> 0 and `bad`) and linear cell id of one particle
__device__ __forceinline__ unsigned int wrap_cell(float &x, float &y, float &z, const Grid &g, bool &bad)
{
    if (!(isfinite(x) && isfinite(y) && isfinite(z))) { bad = true; x = y = z = 0.0f; }
    x = wrap1(x, g.L);
    y = wrap1(y, g.L);
    z = wrap1(z, g.L);
    return cell_id(cell1(x, g), cell1(y, g), cell1(z, g), g.n);
}

// Walks the particles [i0, i1) of one CTA four at a time: thread t takes the quads t, t + T, ...
// With VEC (pos 16-byte aligned, i0 a multiple of 4) a quad is three 128-bit loads, all issued
// before the first use, so every thread keeps 48 bytes in flight; f(x, y, z, i) is called per particle.
template <bool VEC, int THREADS, typename F>
__device__ __forceinline__ void for_each_particle(const float *__restrict__ pos, int64_t i0, int64_t i1, F f)
{
    for (int64_t i = i0 + 4 * (int64_t)threadIdx.x; i < i1; i += 4 * (int64_t)THREADS) {
        if (VEC && i + 4 <= i1) {
            const float4 *q = reinterpret_cast<const float4 *>(pos + 3 * i);
            const float4 a = __ldg(q), b = __ldg(q + 1), c = __ldg(q + 2);
            f(a.x, a.y, a.z, i);
            f(a.w, b.x, b.y, i + 1);
            f(b.z, b.w, c.x, i + 2);
            f(c.y, c.z, c.w, i + 3);
        } else {
            const int m = (int)min((int64_t)4, i1 - i);
            float v[12];
#pragma unroll
            for (int k = 0; k < 12; ++k) v[k] = (k < 3 * m) ? __ldg(pos + 3 * i + k) : 0.0f;
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (k < m) f(v[3 * k], v[3 * k + 1], v[3 * k + 2], i + k);
        }
    }
}

// ---- link predicate (north_star's single float32 expression):
// per axis d = wi - wj; d > h ? d - L : (d < -h ? d + L : d);  d2 = (dx dx + dy dy) + dz dz <= b2.
__device__ __forceinline__ float min_image(float d, float L, float h)
{
    if (d > h) d = __fsub_rn(d, L);
    else if (d < -h) d = __fadd_rn(d, L);
    return d;
}

__device__ __forceinline__ bool linked(float xi, float yi, float zi, float xj, float yj, float zj, const Grid &g)
{
    float dx = min_image(__fsub_rn(xi, xj), g.L, g.h);
    float dy = min_image(__fsub_rn(yi, yj), g.L, g.h);
    float dz = min_image(__fsub_rn(zi, zj), g.L, g.h);
    float d2 = __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
    return d2 <= g.b2;
}

// ---- union-find on `rel`: rel[s] = s - parent(s) as a signed offset (a root has rel 0, which
// cell_sort_kernel writes for every slot).  The root of a set is its member with the smallest
// ORIGINAL index (`idx`), i.e. the canonical label of PAPER.md:91 / 180 itself, so H5 needs no
// minimum pass: a root hooks under another one only if its original index is the larger of the
// two (a strict total order: no cycles).  Hooks are atomicCAS(rel + root, 0, offset) and can only
// succeed on a true root; every plain load may return a stale value, which is always the offset
// to SOME ancestor (links only ever move up), so staleness costs hops, never correctness.  Plain
// path-halving stores at non-roots are benign.
__device__ __forceinline__ int find_rel(unsigned int *rel, int x)
{
    int d = (int)rel[x];
    while (d) {
        const int p = x - d;
        const int dp = (int)rel[p];
        if (dp) rel[x] = (unsigned int)(d + dp);  // halve: x -> grandparent
        x = p;
        d = dp;
    }
    return x;
}

__device__ __forceinline__ int unite_rel(unsigned int *rel, const int *__restrict__ idx, int a, int b)
{
    int ra = find_rel(rel, a), rb = find_rel(rel, b);
    while (ra != rb) {
        if (__ldg(idx + ra) < __ldg(idx + rb)) { const int t = ra; ra = rb; rb = t; }  // ra: larger original index
        const unsigned int old = atomicCAS(rel + ra, 0u, (unsigned int)(ra - rb));
        if (old == 0u) return rb;
        ra = find_rel(rel, ra - (int)old);
    }
    return ra;
}

__device__ __forceinline__ unsigned long long ld_relaxed_u64(const unsigned long long *p)
{
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ void st_relaxed_u64(unsigned long long *p, unsigned long long v)
{
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// Brackets one profiled stage (fof_profile_*) around the launches of a multi-kernel launcher.
struct StageHook {
    fof_handle *h;
    cudaStream_t s;
    int base;  // stage id of the launcher's first kernel
    void begin(int k, int kernels);
    void end(int k);
};

// kernels (one launcher per step; all asynchronous on `s`)
cudaError_t launch_sort(const float *pos, int64_t N, Grid g, const SortPlan &sp, int ctas, unsigned int *cta_hist,
                        unsigned int *bin_base, float4 *part, unsigned int *cell_start, float4 *sorted,
                        unsigned int *rel, int *idx_s, unsigned long long *dense_list, int *labels, Ctrl *ctrl,
                        const unsigned int *gate, int *cnt, StageHook &hook, cudaStream_t s);
// block path (kernels_block.cu): histogram + offsets + partition into blocks (with ghost copies), one CTA per
// block links out of shared memory, equivalence pairs across blocks, flatten.  Sets ctrl->mode = 1 (and does
// nothing else) if a block does not fit: the gated cell path then runs instead.
cudaError_t launch_block_path(const float *pos, int64_t N, Grid g, const BlockGeom &bg, int ctas, unsigned int *cursor,
                              float4 *part, int2 *cross, int *labels, int *cnt, unsigned long long *state,
                              int64_t state_items, Ctrl *ctrl, StageHook &hook, cudaStream_t s);
cudaError_t launch_link(const float4 *sorted, int64_t N, Grid g, const unsigned int *cell_start,
                        const unsigned long long *dense_list, unsigned int *rel, const int *idx_s, Ctrl *ctrl,
                        int num_sms, const unsigned int *gate, cudaStream_t s);
cudaError_t launch_grid_pairs(const unsigned int *cell_start, Grid g, Ctrl *ctrl, int num_sms, cudaStream_t s);
cudaError_t launch_write_labels(const unsigned int *rel, const int *idx_s, int *labels, int64_t N,
                                const unsigned int *gate, int *cnt, unsigned long long *state, int64_t state_items,
                                Ctrl *ctrl, cudaStream_t s);

cudaError_t launch_group_count(const int *labels, int64_t N, int *cnt, unsigned long long *state,
                               int64_t state_items, Ctrl *ctrl, cudaStream_t s);
cudaError_t launch_group_compact(const int *labels, int64_t N, int N_min, int *cnt_to_gid, int64_t cap,
                                 int *group_label, int *group_size, double *acc, unsigned long long *state,
                                 Ctrl *ctrl, int64_t tiles, cudaStream_t s);
cudaError_t launch_group_reduce(const float *pos, const float *mass, const int *labels, int64_t N, Grid g,
                                const int *gid, int64_t cap, const int *group_size, double *acc, int *particle_group,
                                cudaStream_t s);
cudaError_t launch_group_finish(const float *pos, const int *group_label, const int *group_size,
                                const double *acc, bool has_mass, Grid g, int64_t cap, const Ctrl *ctrl,
                                float *group_mass, float *group_com, cudaStream_t s);


cudaError_t launch_group_sigma(const float *pos, const float *mass, const int *particle_group, int64_t N, Grid g,
                               const float *group_mass, const float *group_com, int64_t K, double *acc,
                               float *group_sigma, cudaStream_t s);
cudaError_t launch_groups_backward(const float *pos, const float *mass, const int *particle_group, int64_t N, Grid g,
                                   const float *group_mass, const float *group_com, const float *group_sigma,
                                   const float *grad_com, const float *grad_sigma, int64_t K, float *grad_pos,
                                   cudaStream_t s);

cudaError_t launch_link_stochastic(const float4 *sorted, int64_t N, Grid g, const unsigned int *cell_start,
                                   const int *idx_s, unsigned int *rel, float b_link, float alpha,
                                   unsigned long long seed, unsigned int sample, int *labels, double *logp, float *grad,
                                   Ctrl *ctrl, cudaStream_t s);
cudaError_t launch_link_stochastic_batch(const float4 *sorted, int64_t N, Grid g, const unsigned int *cell_start,
                                         const int *idx_s, unsigned int *rel_s, float b_link, float alpha,
                                         unsigned long long seed, unsigned int sample0, int S, int *labels,
                                         double *logp, float *grad, Ctrl *ctrl, cudaStream_t s);

// The potential-edge list of the stochastic path (fof_stochastic_list_build): views into the caller's buffer.
struct StochListHead {
    unsigned long long records;    // directed records (every potential edge appears under both of its particles)
    unsigned long long potential;  // potential edges (owned records)
    double logp0;                  // log p(y = 0): sum over the potential edges of log(1 - p)
};
constexpr int kListScanTile = 4096;  // entries per CTA of the offset scan
struct StochList {
    StochListHead *head;
    unsigned long long *bsum;  // per scan tile: entries before it
    unsigned int *roff;        // [N + 1] first record of every home particle (cell-sorted slot order)
    int *home_orig;            // [N] original index of the home particle
    uint4 *rec;                // two uint4 per record
};
inline size_t stoch_list_align(size_t x) { return (x + 255) & ~(size_t)255; }
inline size_t stoch_list_fixed_bytes(int64_t N)
{
    const size_t tiles = (size_t)((N + kListScanTile) / kListScanTile) + 1;
    return 256 + stoch_list_align(tiles * 8) + stoch_list_align(((size_t)N + 1) * 4) + stoch_list_align((size_t)N * 4 + 4);
}
inline StochList stoch_list_views(void *list, int64_t N)
{
    const size_t tiles = (size_t)((N + kListScanTile) / kListScanTile) + 1;
    char *p = static_cast<char *>(list);
    StochList v;
    v.head = (StochListHead *)p;          p += 256;
    v.bsum = (unsigned long long *)p;     p += stoch_list_align(tiles * 8);
    v.roff = (unsigned int *)p;           p += stoch_list_align(((size_t)N + 1) * 4);
    v.home_orig = (int *)p;               p += stoch_list_align((size_t)N * 4 + 4);
    v.rec = (uint4 *)p;
    return v;
}
cudaError_t launch_stoch_list_count(const float4 *sorted, int64_t N, Grid g, const unsigned int *cell_start,
                                    const int *idx_s, unsigned int *counts, cudaStream_t s);
cudaError_t launch_stoch_list_offsets(const unsigned int *counts, int64_t N, StochList list, cudaStream_t s);
cudaError_t launch_stoch_list_fill(const float4 *sorted, int64_t N, Grid g, const unsigned int *cell_start,
                                   const int *idx_s, float b_link, float alpha, StochList list, cudaStream_t s);
cudaError_t launch_link_stochastic_list(StochList list, int64_t N, float b_link, float alpha, unsigned long long seed,
                                        unsigned int sample0, int S, unsigned int *rel_s, int *labels, double *logp,
                                        float *grad, Ctrl *ctrl, int num_sms, cudaStream_t s);

cudaError_t launch_subgroups(const float *pos, const float *vel, const int *particle_group, const int *group_size,
                             int64_t N, int64_t K, float L, float sigma_x, float sigma_v, float ell,
                             unsigned int *offsets, unsigned int *cursor, int *members, unsigned int *sub_rel,
                             int *sub_labels, Ctrl *ctrl, int num_sms, cudaStream_t s);

cudaError_t launch_layer_select(const float *pos, int64_t N, float L, int axis, float lo, float width, int *out_idx,
                                unsigned int *count, cudaStream_t s);
cudaError_t launch_component_min(const int *labels, const int *ids, int64_t N, int *tmp, int *out, cudaStream_t s);
cudaError_t launch_merge_labels(const int *pairs, int64_t P, int *parent, int64_t G, int *labels, int64_t N,
                                cudaStream_t s);
cudaError_t launch_merge_labels_sparse(const int *pairs, int64_t P, const int *uniq, int64_t U, int *parent, int *labels,
                                       int64_t N, cudaStream_t s);
cudaError_t launch_combine_groups(const int *want, int64_t W, const float *ref, float L, const int *part_label, int64_t P,
                                  const int *part_size, const float *part_mass, const float *part_com, int *out_size,
                                  float *out_mass, float *out_com, cudaStream_t s);

}  // namespace fof
