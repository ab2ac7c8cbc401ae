// fof_api.cu — the C ABI declared in include/fof.h: plan (H0), workspace layout, call sequencing.
// No device memory is allocated here; every step of the path runs in the kernels of this library.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "fof_internal.cuh"

using namespace fof;

namespace {
// Most work items the cell sort can list: every dense cell of m particles gives at most m / kDenseCell
// tiles, a heavy one (m >= kHeavyCell) at most (m / 32 + 1) kHeavyParts items.
size_t dense_items_max(size_t N)
{
    const size_t plain = N / kDenseCell, heavy = (N / 32 + N / kHeavyCell + 1) * kHeavyParts;
    return (plain > heavy ? plain : heavy) + 2;
}


inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

constexpr bool kAutoIsBlocks = false;  // what FOF_PATH_AUTO means where the plan admits the block path

// H0, block path: blocks of 2^sx x 2^sy x 2^sz cells with >= 3 blocks per axis (so that the forward and the
// backward neighbour of a block are different blocks), at most kMaxBlockBins blocks, and a mean occupancy of
// about half of what block_link_kernel holds (kBlockCap records, own + ghost copies).
void plan_blocks(fof_handle *h)
{
    h->block_ok = false;
    BlockGeom &bg = h->bg;
    memset(&bg, 0, sizeof(bg));
    if (h->N <= 0 || h->n < 6) return;
    int smax = 0;
    while ((2 << smax) <= (h->n - 1) / 2) ++smax;  // largest s with ceil(n / 2^s) >= 3
    if (((h->n + (1 << smax) - 1) >> smax) < 3) return;
    int s[3] = {smax < 4 ? smax : 4, smax < 4 ? smax : 4, smax < 3 ? smax : 3};
    const double rho = (double)h->N / ((double)h->n * h->n * h->n);
    const double target = 0.55 * kBlockCap;
    while ((double)(1 << (s[0] + s[1] + s[2])) * rho > target) {
        int a = 2;  // shrink the longest side, z first
        if (s[1] > s[a]) a = 1;
        if (s[0] > s[a]) a = 0;
        if (s[a] == 0) return;
        --s[a];
    }
    if (s[0] < 1 || s[1] < 1 || s[2] < 1) return;  // blocks one cell wide would be mostly ghosts
    bg.sx = s[0]; bg.sy = s[1]; bg.sz = s[2];
    bg.nbx = (h->n + (1 << bg.sx) - 1) >> bg.sx;
    bg.nby = (h->n + (1 << bg.sy) - 1) >> bg.sy;
    bg.nbz = (h->n + (1 << bg.sz) - 1) >> bg.sz;
    const int64_t bins = (int64_t)bg.nbx * bg.nby * bg.nbz;
    if (bins > kMaxBlockBins) return;
    bg.bins = (int)bins;
    bg.X = (1 << bg.sx) + 2; bg.Y = (1 << bg.sy) + 2; bg.Z = (1 << bg.sz) + 1;
    bg.ncell = bg.X * bg.Y * bg.Z;
    h->block_ok = true;
}

// H0: workspace layout for the current grid.
void layout(fof_handle *h)
{
    const size_t N = (size_t)h->N;
    h->C = (int64_t)h->n * h->n * h->n;
    const int64_t cell_items = h->C + 1;
    h->sort.shift = kMinShift;
    while (((h->C + ((int64_t)1 << h->sort.shift) - 1) >> h->sort.shift) > kMaxBins) ++h->sort.shift;
    h->sort.bins = (int)((h->C + ((int64_t)1 << h->sort.shift) - 1) >> h->sort.shift);
    h->gscan_tiles = h->N > 0 ? (h->N + kScanTile - 1) / kScanTile : 1;
    h->max_groups = h->N / h->N_min;
    plan_blocks(h);
    size_t off = 0;
    h->off_ctrl = off;        off += 256;
    h->off_cell = off;        off += align256(((size_t)cell_items + 8) * sizeof(unsigned int));
    h->off_rel = off;         off += align256((N + 1) * sizeof(unsigned int));
    h->off_cta_hist = off;    off += align256((size_t)kMaxPartCtas * h->sort.bins * sizeof(unsigned int));
    // fine bin offsets, and behind them the coarse ones of the two-pass partition (<= bins / 64 + 2 entries)
    h->off_bin_base = off;    off += align256(((size_t)h->sort.bins + 2 + (size_t)h->sort.bins / 64 + 4) * sizeof(unsigned int));
    // `part` and `sorted` are adjacent: the block path's record array (one slice of kBlockCap records per block)
    // spans both; the cross-block equivalence pairs of the block path live in the idx_s array
    h->off_part = off;        off += align256((N + 1) * sizeof(float4));
    h->off_sorted = off;      off += align256((N + 1) * sizeof(float4));
    if (h->block_ok) {  // the block path's fixed slices: bins x kBlockCap records from off_part on
        const size_t need = h->off_part + align256((size_t)h->bg.bins * kBlockCap * sizeof(float4));
        if (need > off) off = need;
    }
    h->off_idx = off;         off += align256((2 * N + 2) * sizeof(int));  // also: one int2 per linked ghost record
    h->off_dense = off;       off += align256(dense_items_max(N) * sizeof(unsigned long long));
    h->off_cursor = off;      off += align256(((size_t)kMaxBlockBins + 2) * sizeof(unsigned int));
    h->off_cnt = off;         off += align256((N + 1) * sizeof(int));
    h->off_acc = off;         off += align256(((size_t)h->max_groups + 1) * 4 * sizeof(double));
    h->off_gscan_state = off; off += align256((size_t)h->gscan_tiles * sizeof(unsigned long long));
    h->ws_bytes = off;
    h->grid.L = h->L;
    h->grid.h = 0.5f * h->L;
    h->grid.b2 = h->b * h->b;  // host float multiply: one rounding, no FMA possible
    h->grid.inv_cell = (float)((double)h->n / (double)h->L);
    h->grid.n = h->n;
    h->grid.n_minus_1 = h->n - 1;
    // reach filter: b in cell units, plus 1e-3 cells and the float32 resolution of a position in
    // cell units (n * 2^-20, several ulp of L), rounded up
    h->grid.reach = nextafterf((float)((double)h->b * (double)h->n / (double)h->L + 1e-3 +
                                       (double)h->n * 9.5367431640625e-07), 2.0f);
    h->linked = false;
    h->linked_ws = nullptr;
    h->counted = false;
}

int cuda_fail(fof_handle *h, cudaError_t e, const char *where)
{
    snprintf(h->cuda_err, sizeof(h->cuda_err), "%s: %s", where, cudaGetErrorString(e));
    (void)cudaGetLastError();
    return FOF_ERR_CUDA;
}

#define CK(call, where)                                   \
    do {                                                  \
        cudaError_t e__ = (call);                         \
        if (e__ != cudaSuccess) return cuda_fail(h, e__, where); \
    } while (0)

// Profiled stages, in execution order (fof_profile_name).
enum Stage { kLinkClear = 0, kBlockPartition, kBlockLink, kBlockCross, kBlockFlatten,
             kLinkHist, kLinkOffsets, kLinkPartition, kLinkCellSort, kLinkPairs, kLinkLabels,
             kGroupsClear, kGroupsCount, kGroupsCompact, kGroupsReduce, kGroupsFinish, kNumStages };
const char *const kStageName[kNumStages] = {
    "link.clear", "block.partition", "block.link", "block.cross", "block.flatten",
    "link.hist", "link.offsets", "link.partition", "link.cell_sort", "link.pairs", "link.labels",
    "groups.clear", "groups.count", "groups.compact", "groups.reduce", "groups.finish"};
static_assert(kNumStages <= kMaxStages, "raise kMaxStages");

struct StageTimer {  // records the two events of a stage around its launches
    fof_handle *h; cudaStream_t s; int k;
    StageTimer(fof_handle *h_, cudaStream_t s_, int k_, int kernels) : h(h_), s(s_), k(k_)
    {
        h->launches += (unsigned long long)kernels;
        if (on()) {
            cudaEventRecord(h->ev[(h->prof_cur * kMaxStages + k) * 2], s);
            h->ev_valid[h->prof_cur * kMaxStages + k] = true;
        }
    }
    ~StageTimer() { if (on()) cudaEventRecord(h->ev[(h->prof_cur * kMaxStages + k) * 2 + 1], s); }
    bool on() const { return h->prof_slots && (h->prof_only < 0 || h->prof_only == k); }
};

}  // namespace

namespace fof {
void StageHook::begin(int k, int kernels)
{
    h->launches += (unsigned long long)kernels;
    if (h->prof_slots && (h->prof_only < 0 || h->prof_only == base + k)) {
        cudaEventRecord(h->ev[(h->prof_cur * kMaxStages + base + k) * 2], s);
        h->ev_valid[h->prof_cur * kMaxStages + base + k] = true;
    }
}
void StageHook::end(int k)
{
    if (h->prof_slots && (h->prof_only < 0 || h->prof_only == base + k))
        cudaEventRecord(h->ev[(h->prof_cur * kMaxStages + base + k) * 2 + 1], s);
}
}  // namespace fof

namespace {

template <typename T>
inline T *at(void *ws, size_t off) { return reinterpret_cast<T *>(static_cast<char *>(ws) + off); }

}  // namespace

extern "C" {

float fof_linking_length(float b_frac, float L, int64_t N)
{
    if (N <= 0) return 0.0f;
    return (float)((double)b_frac * (double)L / cbrt((double)N));
}

int fof_create(int64_t N, float L, float b, int32_t N_min, fof_handle **out)
{
    if (!out) return FOF_ERR_INVALID_ARG;
    if (N < 0 || N > 2147483647LL - 1024) return FOF_ERR_INVALID_ARG;
    if (!(L > 0.0f) || !(b > 0.0f) || !isfinite(L) || !isfinite(b) || N_min < 1) return FOF_ERR_INVALID_ARG;
    // largest grid whose cell side L/n is >= b * kCellMargin (PAPER.md:194 with the safe rounding)
    double nm = floor((double)L / ((double)b * (double)kCellMargin));
    if (nm < 3.0) return FOF_ERR_UNSUPPORTED;
    int32_t n_max = nm > (double)kMaxGrid ? kMaxGrid : (int32_t)nm;
    // about one cell per particle keeps the cell arrays as small as the particle arrays
    int32_t n_occ = (int32_t)floor(cbrt((double)(N > 27 ? N : 27)) + 1e-9);
    fof_handle *h = new (std::nothrow) fof_handle();
    if (!h) return FOF_ERR_INVALID_ARG;
    memset(h, 0, sizeof(*h));
    h->N = N; h->L = L; h->b = b; h->N_min = N_min;
    h->prof_only = -1;
    h->path = FOF_PATH_AUTO;
    h->n_max = n_max;
    h->n = n_occ < n_max ? n_occ : n_max;
    if (h->n < 3) h->n = 3;
    h->num_sms = 0;
    layout(h);
    *out = h;
    return FOF_OK;
}

static void host_streams_free(fof_handle *h);

void fof_destroy(fof_handle *h)
{
    if (!h) return;
    fof_profile_enable(h, 0);
    if (h->copy_stream) {
        (void)cudaStreamDestroy(h->copy_stream);
        (void)cudaEventDestroy(h->ev_linked);
    }
    if (h->in_stream) {
        (void)cudaDeviceSynchronize();  // a submitted input may still be in flight
        host_streams_free(h);
    }
    delete h;
}

int fof_profile_enable(fof_handle *h, int slots)
{
    if (!h || slots < 0 || slots > 1024) return FOF_ERR_INVALID_ARG;
    if (h->prof_slots) {
        const int n = h->prof_slots * kMaxStages * 2;
        h->prof_slots = 0;
        for (int k = 0; k < n; ++k) (void)cudaEventDestroy(h->ev[k]);
        delete[] h->ev; delete[] h->ev_valid;
        h->ev = nullptr; h->ev_valid = nullptr;
    }
    if (slots) {
        const int n = slots * kMaxStages * 2;
        h->ev = new (std::nothrow) cudaEvent_t[n];
        h->ev_valid = new (std::nothrow) bool[slots * kMaxStages]();
        if (!h->ev || !h->ev_valid) {
            delete[] h->ev; delete[] h->ev_valid;
            h->ev = nullptr; h->ev_valid = nullptr;
            return FOF_ERR_INVALID_ARG;
        }
        for (int k = 0; k < n; ++k) {
            const cudaError_t e = cudaEventCreate(&h->ev[k]);
            if (e != cudaSuccess) {  // give back what was created
                for (int j = 0; j < k; ++j) (void)cudaEventDestroy(h->ev[j]);
                delete[] h->ev; delete[] h->ev_valid;
                h->ev = nullptr; h->ev_valid = nullptr;
                return cuda_fail(h, e, "cudaEventCreate");
            }
        }
        h->prof_cur = slots - 1;
        h->prof_slots = slots;
    }
    return FOF_OK;
}

int fof_profile_only(fof_handle *h, int stage)
{
    if (!h || stage < -1 || stage >= kNumStages) return FOF_ERR_INVALID_ARG;
    h->prof_only = stage;
    return FOF_OK;
}

int fof_profile_count(const fof_handle *) { return kNumStages; }

const char *fof_profile_name(const fof_handle *, int k) { return (k >= 0 && k < kNumStages) ? kStageName[k] : ""; }

int fof_profile_read(fof_handle *h, float *ms, int cap)
{
    if (!h || !ms || cap < 0) return FOF_ERR_INVALID_ARG;
    if (!h->prof_slots) return FOF_ERR_STATE;
    for (int k = 0; k < kNumStages && k < cap; ++k) {
        double sum = 0.0;
        int cnt = 0;
        for (int sl = 0; sl < h->prof_slots; ++sl) {
            const int e = sl * kMaxStages + k;
            if (!h->ev_valid[e]) continue;
            float t = 0.0f;
            CK(cudaEventSynchronize(h->ev[2 * e + 1]), "cudaEventSynchronize");
            CK(cudaEventElapsedTime(&t, h->ev[2 * e], h->ev[2 * e + 1]), "cudaEventElapsedTime");
            sum += t;
            ++cnt;
            h->ev_valid[e] = false;
        }
        ms[k] = cnt ? (float)(sum / cnt) : 0.0f;
    }
    return FOF_OK;
}

uint64_t fof_launch_count(const fof_handle *h) { return h ? h->launches : 0; }

int fof_set_grid(fof_handle *h, int32_t n)
{
    if (!h) return FOF_ERR_INVALID_ARG;
    if (n < 3 || n > h->n_max) return FOF_ERR_INVALID_ARG;
    h->n = n;
    layout(h);
    return FOF_OK;
}

int fof_get_grid(const fof_handle *h, int32_t *n, int64_t *cells, int32_t *n_max)
{
    if (!h) return FOF_ERR_INVALID_ARG;
    if (n) *n = h->n;
    if (cells) *cells = h->C;
    if (n_max) *n_max = h->n_max;
    return FOF_OK;
}

size_t fof_workspace_bytes(const fof_handle *h) { return h ? h->ws_bytes : 0; }

int fof_set_path(fof_handle *h, int32_t path)
{
    if (!h || (path != FOF_PATH_AUTO && path != FOF_PATH_CELLS && path != FOF_PATH_BLOCKS)) return FOF_ERR_INVALID_ARG;
    h->path = path;
    h->linked = false;
    return FOF_OK;
}

int fof_link_path(fof_handle *h, void *ws, void *stream, int32_t *path_host, int32_t *blocks_host,
                  int32_t *max_block_host)
{
    if (!h || !ws) return FOF_ERR_INVALID_ARG;
    if (!h->linked || h->linked_ws != ws) return FOF_ERR_STATE;
    cudaStream_t s = (cudaStream_t)stream;
    Ctrl c;
    CK(cudaMemcpyAsync(&c, at<Ctrl>(ws, h->off_ctrl), sizeof(Ctrl), cudaMemcpyDeviceToHost, s), "copy ctrl");
    CK(cudaStreamSynchronize(s), "sync");
    const bool blocks = !h->linked_cells && c.mode == 0u;
    if (path_host) *path_host = blocks ? FOF_PATH_BLOCKS : FOF_PATH_CELLS;
    if (blocks_host) *blocks_host = h->block_ok ? h->bg.bins : 0;
    if (max_block_host) *max_block_host = h->linked_cells ? 0 : (int32_t)c.max_block;
    return FOF_OK;
}

int fof_link(fof_handle *h, const float *pos, int32_t *labels, void *ws, void *stream)
{
    if (!h || !ws || ((uintptr_t)ws & 255)) return FOF_ERR_INVALID_ARG;
    if (h->N > 0 && (!pos || !labels)) return FOF_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    if (h->num_sms == 0) {
        int dev = 0, sms = 0;
        CK(cudaGetDevice(&dev), "cudaGetDevice");
        CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev), "cudaDeviceGetAttribute");
        h->num_sms = sms;
    }
    // level-1 partition: one CTA of 1024 threads per SM (measured: fewer open write streams beat occupancy)
    h->part_ctas = h->num_sms < kMaxPartCtas ? h->num_sms : kMaxPartCtas;
    Ctrl *ctrl = at<Ctrl>(ws, h->off_ctrl);
    unsigned int *cell = at<unsigned int>(ws, h->off_cell);
    float4 *sorted = at<float4>(ws, h->off_sorted);
    unsigned int *rel = at<unsigned int>(ws, h->off_rel);
    int *idx_s = at<int>(ws, h->off_idx);
    unsigned long long *dense = at<unsigned long long>(ws, h->off_dense);
    h->linked = false;
    h->counted = false;
    const int has = h->N > 0;
    int *cnt = at<int>(ws, h->off_cnt);
    unsigned long long *gstate = at<unsigned long long>(ws, h->off_gscan_state);
    if (h->prof_slots) {
        h->prof_cur = (h->prof_cur + 1) % h->prof_slots;
        for (int k = 0; k < kNumStages; ++k) h->ev_valid[h->prof_cur * kMaxStages + k] = false;
    }
    {   // only the control block needs clearing: every other array is fully written by the sort
        StageTimer t(h, s, kLinkClear, 0);
        CK(cudaMemsetAsync(ctrl, 0, 256, s), "memset ctrl");
    }
    // Block path first where the plan admits it; it leaves ctrl->mode = 1 (and nothing else) when a block does
    // not fit shared memory, and the cell path below, gated on that flag, then does the work.
    const bool blocks = h->block_ok && (h->path == FOF_PATH_BLOCKS || (h->path == FOF_PATH_AUTO && kAutoIsBlocks)) && has;
    if (blocks) {
        StageHook hook{h, s, kBlockPartition};
        CK(launch_block_path(pos, h->N, h->grid, h->bg, h->part_ctas, at<unsigned int>(ws, h->off_cursor),
                             at<float4>(ws, h->off_part), at<int2>(ws, h->off_idx), labels, cnt, gstate, h->gscan_tiles, ctrl,
                             hook, s),
           "block path kernels");
    }
    const unsigned int *gate = blocks ? &ctrl->mode : nullptr;
    {
        StageHook hook{h, s, kLinkHist};
        CK(launch_sort(pos, h->N, h->grid, h->sort, h->part_ctas, at<unsigned int>(ws, h->off_cta_hist),
                       at<unsigned int>(ws, h->off_bin_base), at<float4>(ws, h->off_part), cell, sorted, rel, idx_s,
                       dense, labels, ctrl, gate, cnt, hook, s), "sort kernels");
    }
    {
        StageTimer t(h, s, kLinkPairs, has);
        CK(launch_link(sorted, h->N, h->grid, cell, dense, rel, idx_s, ctrl, h->num_sms, gate, s), "link kernels");
    }
    {
        StageTimer t(h, s, kLinkLabels, has);
        CK(launch_write_labels(rel, idx_s, labels, h->N, gate, cnt, gstate, h->gscan_tiles, ctrl, s), "write_labels_kernel");
    }
    h->linked = true;
    h->linked_ws = ws;
    h->slist = nullptr;  // a potential-edge list describes the positions of the link it was built after
    h->slist_counts_ws = nullptr;
    h->counted = has != 0;  // H6 rode along: fof_groups on these very labels starts at the compaction
    h->counted_labels = labels;
    h->linked_cells = !blocks;  // the cell-sorted arrays are certainly there only if the cell path ran ungated
    return FOF_OK;
}

int fof_link_stats(fof_handle *h, void *ws, void *stream, uint64_t *edges_host, uint64_t *pair_tests_host,
                   uint64_t *grid_pairs_host)
{
    if (!h || !ws) return FOF_ERR_INVALID_ARG;
    if (!h->linked || h->linked_ws != ws) return FOF_ERR_STATE;
    cudaStream_t s = (cudaStream_t)stream;
    Ctrl c;
    Ctrl *ctrl = at<Ctrl>(ws, h->off_ctrl);
    if (grid_pairs_host && h->N > 0 && h->linked_cells) {  // computed on demand from the cell offsets left in the workspace
        CK(cudaMemsetAsync(&ctrl->grid_pairs, 0, sizeof(unsigned long long), s), "memset grid_pairs");
        CK(launch_grid_pairs(at<unsigned int>(ws, h->off_cell), h->grid, ctrl, h->num_sms, s), "grid_pairs_kernel");
    }
    CK(cudaMemcpyAsync(&c, ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, s), "copy ctrl");
    CK(cudaStreamSynchronize(s), "sync");
    const bool blocks = !h->linked_cells && c.mode == 0u;  // the block path did the work: its counters count
    if (edges_host) *edges_host = blocks ? c.edges_b : c.edges;
    if (pair_tests_host) *pair_tests_host = blocks ? c.pair_tests_b : c.pair_tests;
    if (grid_pairs_host) *grid_pairs_host = c.grid_pairs;
    return FOF_OK;
}

}  // extern "C"

// The kernels of fof_groups, enqueued on `s` without waiting for them (fof_groups and fof_host_submit share it):
// K is left in the workspace's Ctrl.
static int groups_enqueue(fof_handle *h, const float *pos, const float *mass, const int32_t *labels, void *ws,
                          int32_t *group_label, int32_t *group_size, float *group_mass, float *group_com,
                          int32_t *particle_group, int64_t cap, cudaStream_t s)
{
    Ctrl *ctrl = at<Ctrl>(ws, h->off_ctrl);
    int *cnt = at<int>(ws, h->off_cnt);
    double *acc = at<double>(ws, h->off_acc);
    unsigned long long *state = at<unsigned long long>(ws, h->off_gscan_state);
    const int has = h->N > 0;
    if (h->prof_slots)
        for (int k = kGroupsClear; k <= kGroupsFinish; ++k) h->ev_valid[h->prof_cur * kMaxStages + k] = false;
    // The sizes of the groups of `labels` are already in the workspace if these are the labels the last fof_link
    // on (h, ws) wrote (H6 is fused into its label pass); any other labels are counted here.
    const bool counted = h->counted && h->linked && h->linked_ws == ws && h->counted_labels == (const void *)labels;
    h->counted = false;  // the compaction below overwrites the counters
    h->slist_counts_ws = nullptr;
    if (!counted) {
        {
            StageTimer t(h, s, kGroupsClear, 0);
            CK(cudaMemsetAsync(cnt, 0, (size_t)(h->N + 1) * sizeof(int), s), "memset cnt");
        }
        {   // also clears the compaction's ticket, K and scan state
            StageTimer t(h, s, kGroupsCount, 1);
            CK(launch_group_count(labels, h->N, cnt, state, h->gscan_tiles, ctrl, s), "group_count_kernel");
        }
    }
    {
        StageTimer t(h, s, kGroupsCompact, has);
        CK(launch_group_compact(labels, h->N, h->N_min, cnt, cap, group_label, group_size, acc, state, ctrl,
                                h->gscan_tiles, s), "group_compact_kernel");
    }
    {
        StageTimer t(h, s, kGroupsReduce, has);
        CK(launch_group_reduce(pos, mass, labels, h->N, h->grid, cnt, cap, group_size, acc, particle_group, s),
           "group_reduce_kernel");
    }
    const int64_t fin = cap < h->max_groups ? cap : h->max_groups;
    {
        StageTimer t(h, s, kGroupsFinish, fin > 0);
        CK(launch_group_finish(pos, group_label, group_size, acc, mass != nullptr, h->grid, fin, ctrl, group_mass,
                               group_com, s), "group_finish_kernel");
    }
    return FOF_OK;
}

extern "C" {

int fof_groups(fof_handle *h, const float *pos, const float *mass, const int32_t *labels, void *ws,
               int32_t *group_label, int32_t *group_size, float *group_mass, float *group_com,
               int32_t *particle_group, int64_t cap, int64_t *K_host, void *stream)
{
    if (!h || !ws || ((uintptr_t)ws & 255) || !K_host || cap < 0) return FOF_ERR_INVALID_ARG;
    if (h->N > 0 && (!pos || !labels)) return FOF_ERR_INVALID_ARG;
    if (cap > 0 && (!group_label || !group_size || !group_mass || !group_com)) return FOF_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    *K_host = 0;
    const int rc = groups_enqueue(h, pos, mass, labels, ws, group_label, group_size, group_mass, group_com,
                                  particle_group, cap, s);
    if (rc != FOF_OK) return rc;
    long long K = 0;
    CK(cudaMemcpyAsync(&K, &at<Ctrl>(ws, h->off_ctrl)->K, sizeof(K), cudaMemcpyDeviceToHost, s), "copy K");
    CK(cudaStreamSynchronize(s), "sync");
    *K_host = (int64_t)K;
    if (K > cap) return FOF_ERR_CAPACITY;
    return FOF_OK;
}

int fof_link_stochastic(fof_handle *h, float b_link, float alpha, uint64_t seed, uint32_t sample, int32_t *labels,
                        double *logp, float *grad_pos, void *ws, void *stream)
{
    if (!h || !ws || ((uintptr_t)ws & 255) || !logp) return FOF_ERR_INVALID_ARG;
    if (!(b_link > 0.0f) || !(b_link <= h->b) || !isfinite(alpha)) return FOF_ERR_INVALID_ARG;
    if (h->N > 0 && !labels) return FOF_ERR_INVALID_ARG;
    if (!h->linked || h->linked_ws != ws || !h->linked_cells) return FOF_ERR_STATE;  // needs the cell sort of a fof_link on (h, ws)
    cudaStream_t s = (cudaStream_t)stream;
    h->counted = false;  // the caller may be overwriting the labels buffer whose group sizes were counted
    h->launches += h->N > 0 ? 3 : 0;
    CK(launch_link_stochastic(at<float4>(ws, h->off_sorted), h->N, h->grid, at<unsigned int>(ws, h->off_cell),
                              at<int>(ws, h->off_idx), at<unsigned int>(ws, h->off_rel), b_link, alpha, seed, sample,
                              labels, logp, grad_pos, at<Ctrl>(ws, h->off_ctrl), s), "stochastic link kernels");
    return FOF_OK;
}

size_t fof_stochastic_scratch_bytes(const fof_handle *h, int32_t S)
{
    if (!h || S <= 0) return 0;
    return (size_t)S * ((size_t)h->N + 1) * sizeof(unsigned int);
}

int fof_link_stochastic_batch(fof_handle *h, float b_link, float alpha, uint64_t seed, uint32_t sample0, int32_t S,
                              int32_t *labels, double *logp, float *grad_pos, void *scratch, void *ws, void *stream)
{
    if (!h || !ws || ((uintptr_t)ws & 255) || !logp || S <= 0 || S > 1024) return FOF_ERR_INVALID_ARG;
    if (!(b_link > 0.0f) || !(b_link <= h->b) || !isfinite(alpha)) return FOF_ERR_INVALID_ARG;
    if (h->N > 0 && (!labels || !scratch || ((uintptr_t)scratch & 3))) return FOF_ERR_INVALID_ARG;
    if (!h->linked || h->linked_ws != ws || !h->linked_cells) return FOF_ERR_STATE;  // needs the cell sort of a fof_link on (h, ws)
    cudaStream_t s = (cudaStream_t)stream;
    h->counted = false;
    h->launches += h->N > 0 ? (unsigned long long)(S / 4 + S % 4 + 2 * S) : 0;
    CK(launch_link_stochastic_batch(at<float4>(ws, h->off_sorted), h->N, h->grid, at<unsigned int>(ws, h->off_cell),
                                    at<int>(ws, h->off_idx), static_cast<unsigned int *>(scratch), b_link, alpha, seed,
                                    sample0, S, labels, logp, grad_pos, at<Ctrl>(ws, h->off_ctrl), s),
       "stochastic link kernels (batch)");
    return FOF_OK;
}

size_t fof_stochastic_list_bytes(const fof_handle *h, uint64_t records)
{
    if (!h) return 0;
    return stoch_list_fixed_bytes(h->N) + (size_t)records * 32;
}

int fof_stochastic_list_build(fof_handle *h, float b_link, float alpha, void *list, size_t list_bytes,
                              uint64_t *records_host, void *ws, void *stream)
{
    if (!h || !ws || ((uintptr_t)ws & 255) || !list || ((uintptr_t)list & 255) || !records_host) return FOF_ERR_INVALID_ARG;
    if (!(b_link > 0.0f) || !(b_link <= h->b) || !isfinite(alpha)) return FOF_ERR_INVALID_ARG;
    if (list_bytes < stoch_list_fixed_bytes(h->N)) return FOF_ERR_INVALID_ARG;
    if (!h->linked || h->linked_ws != ws || !h->linked_cells) return FOF_ERR_STATE;  // needs the cell sort of a fof_link on (h, ws)
    cudaStream_t s = (cudaStream_t)stream;
    const StochList v = stoch_list_views(list, h->N);
    h->slist = nullptr;
    *records_host = 0;
    // The record counts of every particle go to the workspace (the group-size counters, free between fof_link and
    // fof_groups) and stay valid until one of those runs: the call that sizes the buffer pays for the search, the
    // call that fills it does not search again.
    unsigned int *counts = reinterpret_cast<unsigned int *>(at<int>(ws, h->off_cnt));
    h->counted = false;
    if (h->slist_counts_ws != ws) {
        h->launches += h->N > 0 ? 1 : 0;
        CK(launch_stoch_list_count(at<float4>(ws, h->off_sorted), h->N, h->grid, at<unsigned int>(ws, h->off_cell),
                                   at<int>(ws, h->off_idx), counts, s), "stochastic list: count");
        h->slist_counts_ws = ws;
    }
    h->launches += 3;
    CK(launch_stoch_list_offsets(counts, h->N, v, s), "stochastic list: offsets");
    StochListHead head;
    CK(cudaMemcpyAsync(&head, v.head, sizeof(head), cudaMemcpyDeviceToHost, s), "copy list head");
    CK(cudaStreamSynchronize(s), "sync");
    *records_host = (uint64_t)head.records;
    if (head.records > 0xffffffffull || list_bytes < fof_stochastic_list_bytes(h, head.records)) return FOF_ERR_CAPACITY;
    h->launches += h->N > 0 ? 1 : 0;
    CK(launch_stoch_list_fill(at<float4>(ws, h->off_sorted), h->N, h->grid, at<unsigned int>(ws, h->off_cell),
                              at<int>(ws, h->off_idx), b_link, alpha, v, s), "stochastic list: fill");
    h->slist = list;
    h->slist_b_link = b_link;
    h->slist_alpha = alpha;
    return FOF_OK;
}

int fof_link_stochastic_list(fof_handle *h, const void *list, uint64_t seed, uint32_t sample0, int32_t S,
                             int32_t *labels, double *logp, float *grad_pos, void *scratch, void *ws, void *stream)
{
    if (!h || !ws || ((uintptr_t)ws & 255) || !list || !logp || S <= 0 || S > 1024) return FOF_ERR_INVALID_ARG;
    if (h->N > 0 && (!labels || !scratch || ((uintptr_t)scratch & 3))) return FOF_ERR_INVALID_ARG;
    if (!h->slist || h->slist != list) return FOF_ERR_STATE;  // not the list of the last fof_stochastic_list_build
    cudaStream_t s = (cudaStream_t)stream;
    h->counted = false;  // the caller may be overwriting the labels buffer whose group sizes were counted
    h->launches += h->N > 0 ? (unsigned long long)(S / 4 + S % 4 + 2 * S) : 0;
    CK(launch_link_stochastic_list(stoch_list_views(const_cast<void *>(list), h->N), h->N, h->slist_b_link,
                                   h->slist_alpha, seed, sample0, S, static_cast<unsigned int *>(scratch), labels, logp,
                                   grad_pos, at<Ctrl>(ws, h->off_ctrl), h->num_sms, s),  // num_sms: set by the fof_link before the build
       "stochastic link kernels (list)");
    return FOF_OK;
}

int fof_subgroups(fof_handle *h, const float *pos, const float *vel, const int32_t *particle_group,
                  const int32_t *group_size, int64_t K, float sigma_x, float sigma_v, float ell, int32_t *sub_labels,
                  void *ws, void *stream)
{
    if (!h || !ws || ((uintptr_t)ws & 255) || K < 0 || K > h->N) return FOF_ERR_INVALID_ARG;
    if (!(sigma_x > 0.0f) || !(sigma_v > 0.0f) || !(ell > 0.0f)) return FOF_ERR_INVALID_ARG;
    if (h->N > 0 && (!pos || !vel || !particle_group || !sub_labels)) return FOF_ERR_INVALID_ARG;
    if (K > 0 && !group_size) return FOF_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    if (h->num_sms == 0) {
        int dev = 0, sms = 0;
        CK(cudaGetDevice(&dev), "cudaGetDevice");
        CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev), "cudaDeviceGetAttribute");
        h->num_sms = sms;
    }
    h->linked = false;  // the member lists and their union-find re-use the link's arrays
    h->counted = false;
    h->slist_counts_ws = nullptr;
    h->launches += h->N > 0 ? (K > 0 ? 6 : 3) : 0;
    CK(launch_subgroups(pos, vel, particle_group, group_size, h->N, K, h->L, sigma_x, sigma_v, ell,
                        at<unsigned int>(ws, h->off_cnt), at<unsigned int>(ws, h->off_part), at<int>(ws, h->off_idx),
                        at<unsigned int>(ws, h->off_rel), sub_labels, at<Ctrl>(ws, h->off_ctrl), h->num_sms, s),
       "sub-halo kernels");
    return FOF_OK;
}

int fof_layer_select(const float *pos, int64_t N, float L, int32_t axis, float lo, float width, int32_t *out_idx,
                     uint32_t *count, void *stream)
{
    if (N < 0 || !(L > 0.0f) || axis < 0 || axis > 2 || !(width >= 0.0f) || !count) return FOF_ERR_INVALID_ARG;
    if (N > 0 && (!pos || !out_idx)) return FOF_ERR_INVALID_ARG;
    return launch_layer_select(pos, N, L, axis, lo, width, out_idx, count, (cudaStream_t)stream) == cudaSuccess
               ? FOF_OK : FOF_ERR_CUDA;
}

int fof_component_min(const int32_t *labels, const int32_t *ids, int64_t N, int32_t *tmp, int32_t *out, void *stream)
{
    if (N < 0 || (N > 0 && (!labels || !ids || !tmp || !out))) return FOF_ERR_INVALID_ARG;
    return launch_component_min(labels, ids, N, tmp, out, (cudaStream_t)stream) == cudaSuccess ? FOF_OK : FOF_ERR_CUDA;
}

int fof_merge_labels(const int32_t *pairs, int64_t P, int32_t *parent, int64_t G, int32_t *labels, int64_t N,
                     void *stream)
{
    if (P < 0 || G < 0 || N < 0 || (G > 0 && !parent) || (P > 0 && !pairs) || (N > 0 && !labels))
        return FOF_ERR_INVALID_ARG;
    return launch_merge_labels(pairs, P, parent, G, labels, N, (cudaStream_t)stream) == cudaSuccess ? FOF_OK
                                                                                                    : FOF_ERR_CUDA;
}

int fof_merge_labels_sparse(const int32_t *pairs, int64_t P, const int32_t *uniq, int64_t U, int32_t *parent,
                            int32_t *labels, int64_t N, void *stream)
{
    if (P < 0 || U < 0 || N < 0 || U > 2147483647LL || (U > 0 && (!parent || !uniq)) || (P > 0 && !pairs) ||
        (N > 0 && !labels))
        return FOF_ERR_INVALID_ARG;
    return launch_merge_labels_sparse(pairs, P, uniq, U, parent, labels, N, (cudaStream_t)stream) == cudaSuccess
               ? FOF_OK : FOF_ERR_CUDA;
}

int fof_combine_groups(const int32_t *want, int64_t W, const float *ref, float L, const int32_t *part_label, int64_t P,
                       const int32_t *part_size, const float *part_mass, const float *part_com, int32_t *out_size,
                       float *out_mass, float *out_com, void *stream)
{
    if (W < 0 || P < 0 || P > 2147483647LL || !(L > 0.0f)) return FOF_ERR_INVALID_ARG;
    if (W > 0 && (!want || !ref || !out_size || !out_mass || !out_com)) return FOF_ERR_INVALID_ARG;
    if (P > 0 && (!part_label || !part_size || !part_mass || !part_com)) return FOF_ERR_INVALID_ARG;
    return launch_combine_groups(want, W, ref, L, part_label, P, part_size, part_mass, part_com, out_size, out_mass,
                                 out_com, (cudaStream_t)stream) == cudaSuccess ? FOF_OK : FOF_ERR_CUDA;
}

int fof_group_sigma(fof_handle *h, const float *pos, const float *mass, const int32_t *particle_group,
                    const float *group_mass, const float *group_com, int64_t K, void *ws, float *group_sigma,
                    void *stream)
{
    if (!h || !ws || ((uintptr_t)ws & 255) || K < 0 || K > h->max_groups) return FOF_ERR_INVALID_ARG;
    if (h->N > 0 && (!pos || !particle_group)) return FOF_ERR_INVALID_ARG;
    if (K > 0 && (!group_mass || !group_com || !group_sigma)) return FOF_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    h->launches += K > 0 ? 2 : 0;
    CK(launch_group_sigma(pos, mass, particle_group, h->N, h->grid, group_mass, group_com, K,
                          at<double>(ws, h->off_acc), group_sigma, s), "sigma kernels");
    return FOF_OK;
}

int fof_groups_backward(fof_handle *h, const float *pos, const float *mass, const int32_t *particle_group,
                        const float *group_mass, const float *group_com, const float *group_sigma,
                        const float *grad_com, const float *grad_sigma, int64_t K, float *grad_pos, void *stream)
{
    if (!h || K < 0) return FOF_ERR_INVALID_ARG;
    if (h->N > 0 && (!pos || !particle_group || !grad_pos)) return FOF_ERR_INVALID_ARG;
    if (K > 0 && (!group_mass || !group_com)) return FOF_ERR_INVALID_ARG;
    if (grad_sigma && !group_sigma) return FOF_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    h->launches += h->N > 0 ? 1 : 0;
    CK(launch_groups_backward(pos, mass, particle_group, h->N, h->grid, group_mass, group_com, group_sigma, grad_com,
                              grad_sigma, K, grad_pos, s), "groups_backward_kernel");
    return FOF_OK;
}

size_t fof_host_device_bytes(const fof_handle *h, int64_t cap)
{
    if (!h || cap < 0) return 0;
    const size_t N = (size_t)h->N;
    size_t off = 0;
    off += align256((N + 1) * 3 * sizeof(float));  // pos
    off += align256((N + 1) * sizeof(float));      // mass
    off += align256((N + 1) * sizeof(int));        // labels
    off += align256((N + 1) * sizeof(int));        // particle_group
    off += align256(((size_t)cap + 1) * sizeof(int)) * 2;    // group_label, group_size
    off += align256(((size_t)cap + 1) * sizeof(float));      // group_mass
    off += align256(((size_t)cap + 1) * 3 * sizeof(float));  // group_com
    off += h->ws_bytes;
    return off;
}

int fof_run_host(fof_handle *h, const float *pos_host, const float *mass_host, int32_t *labels_host,
                 int32_t *group_label_host, int32_t *group_size_host, float *group_mass_host,
                 float *group_com_host, int32_t *particle_group_host, int64_t cap, int64_t *K_host,
                 void *dev_buf, void *stream)
{
    if (!h || !dev_buf || ((uintptr_t)dev_buf & 255) || !K_host || cap < 0) return FOF_ERR_INVALID_ARG;
    if (h->N > 0 && (!pos_host || !labels_host)) return FOF_ERR_INVALID_ARG;
    if (cap > 0 && (!group_label_host || !group_size_host || !group_mass_host || !group_com_host))
        return FOF_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    const size_t N = (size_t)h->N;
    char *p = static_cast<char *>(dev_buf);
    float *pos = (float *)p;      p += align256((N + 1) * 3 * sizeof(float));
    float *mass = (float *)p;     p += align256((N + 1) * sizeof(float));
    int *labels = (int *)p;       p += align256((N + 1) * sizeof(int));
    int *pgroup = (int *)p;       p += align256((N + 1) * sizeof(int));
    int *glabel = (int *)p;       p += align256(((size_t)cap + 1) * sizeof(int));
    int *gsize = (int *)p;        p += align256(((size_t)cap + 1) * sizeof(int));
    float *gmass = (float *)p;    p += align256(((size_t)cap + 1) * sizeof(float));
    float *gcom = (float *)p;     p += align256(((size_t)cap + 1) * 3 * sizeof(float));
    void *ws = p;
    if (N) CK(cudaMemcpyAsync(pos, pos_host, N * 3 * sizeof(float), cudaMemcpyHostToDevice, s), "H2D pos");
    if (N && mass_host) CK(cudaMemcpyAsync(mass, mass_host, N * sizeof(float), cudaMemcpyHostToDevice, s), "H2D mass");
    int rc = fof_link(h, pos, labels, ws, s);
    if (rc != FOF_OK) return rc;
    // From here on a copy into the caller's labels buffer may be in flight on copy_stream: every return goes
    // through `done`, which waits for it.
    bool copying = false;
    auto done = [&](int code) {
        if (copying) (void)cudaStreamSynchronize(h->copy_stream);
        return code;
    };
#define CKD(call, where)                                          \
    do {                                                          \
        cudaError_t e__ = (call);                                 \
        if (e__ != cudaSuccess) return done(cuda_fail(h, e__, where)); \
    } while (0)
    if (N) {  // the labels travel while the groups are built (fof_groups only reads them)
        if (!h->copy_stream) {
            CKD(cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking), "cudaStreamCreate");
            CKD(cudaEventCreateWithFlags(&h->ev_linked, cudaEventDisableTiming), "cudaEventCreate");
        }
        CKD(cudaEventRecord(h->ev_linked, s), "cudaEventRecord");
        CKD(cudaStreamWaitEvent(h->copy_stream, h->ev_linked, 0), "cudaStreamWaitEvent");
        copying = true;
        CKD(cudaMemcpyAsync(labels_host, labels, N * sizeof(int), cudaMemcpyDeviceToHost, h->copy_stream), "D2H labels");
    }
    rc = fof_groups(h, pos, mass_host ? mass : nullptr, labels, ws, glabel, gsize, gmass, gcom,
                    particle_group_host ? pgroup : nullptr, cap, K_host, s);
    if (rc != FOF_OK) return done(rc);
    const size_t K = (size_t)*K_host;
    if (K) {
        CKD(cudaMemcpyAsync(group_label_host, glabel, K * sizeof(int), cudaMemcpyDeviceToHost, s), "D2H group_label");
        CKD(cudaMemcpyAsync(group_size_host, gsize, K * sizeof(int), cudaMemcpyDeviceToHost, s), "D2H group_size");
        CKD(cudaMemcpyAsync(group_mass_host, gmass, K * sizeof(float), cudaMemcpyDeviceToHost, s), "D2H group_mass");
        CKD(cudaMemcpyAsync(group_com_host, gcom, K * 3 * sizeof(float), cudaMemcpyDeviceToHost, s), "D2H group_com");
    }
    if (N && particle_group_host)
        CKD(cudaMemcpyAsync(particle_group_host, pgroup, N * sizeof(int), cudaMemcpyDeviceToHost, s), "D2H particle_group");
    CKD(cudaStreamSynchronize(s), "sync");
    if (copying) CKD(cudaStreamSynchronize(h->copy_stream), "sync labels copy");
    copying = false;
    Ctrl c;
    CK(cudaMemcpy(&c, at<Ctrl>(ws, h->off_ctrl), sizeof(Ctrl), cudaMemcpyDeviceToHost), "copy ctrl");
    if (c.error & 1u) return FOF_ERR_NONFINITE;
    return FOF_OK;
#undef CKD
}

// The streams, events and pinned control blocks of fof_host_submit / fof_host_wait: created on first use, all or
// nothing (host_streams_free also serves fof_destroy; every member is null until it exists).
static void host_streams_free(fof_handle *h)
{
    for (auto &sl : h->slot) {
        if (sl.out) (void)cudaStreamDestroy(sl.out);
        if (sl.ev_in) (void)cudaEventDestroy(sl.ev_in);
        if (sl.ev_linked) (void)cudaEventDestroy(sl.ev_linked);
        if (sl.ev_groups) (void)cudaEventDestroy(sl.ev_groups);
        if (sl.ev_ctrl) (void)cudaEventDestroy(sl.ev_ctrl);
        if (sl.ctrl_pin) (void)cudaFreeHost(sl.ctrl_pin);
        sl = fof_handle::HostSlot{};
    }
    if (h->in_stream) (void)cudaStreamDestroy(h->in_stream);
    if (h->run_stream) (void)cudaStreamDestroy(h->run_stream);
    h->in_stream = h->run_stream = nullptr;
}

static int host_streams(fof_handle *h)
{
    if (h->in_stream) return FOF_OK;
    cudaError_t e = cudaStreamCreateWithFlags(&h->run_stream, cudaStreamNonBlocking);
    for (auto &sl : h->slot) {
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&sl.out, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&sl.ev_in, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&sl.ev_linked, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&sl.ev_groups, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&sl.ev_ctrl, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaHostAlloc((void **)&sl.ctrl_pin, sizeof(Ctrl), cudaHostAllocDefault);
    }
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&h->in_stream, cudaStreamNonBlocking);  // last: "all exist"
    if (e != cudaSuccess) {
        host_streams_free(h);
        return cuda_fail(h, e, "fof_host_submit: streams");
    }
    return FOF_OK;
}

int fof_host_submit(fof_handle *h, int32_t slot, const float *pos_host, const float *mass_host, int32_t *labels_host,
                    int32_t *group_label_host, int32_t *group_size_host, float *group_mass_host,
                    float *group_com_host, int32_t *particle_group_host, int64_t cap, void *dev_buf)
{
    if (!h || slot < 0 || slot > 1 || !dev_buf || ((uintptr_t)dev_buf & 255) || cap < 0) return FOF_ERR_INVALID_ARG;
    if (h->N > 0 && (!pos_host || !labels_host)) return FOF_ERR_INVALID_ARG;
    if (cap > 0 && (!group_label_host || !group_size_host || !group_mass_host || !group_com_host))
        return FOF_ERR_INVALID_ARG;
    {
        const int rc = host_streams(h);
        if (rc != FOF_OK) return rc;
    }
    fof_handle::HostSlot &sl = h->slot[slot];
    if (sl.busy) return FOF_ERR_STATE;
    const size_t N = (size_t)h->N;
    char *p = static_cast<char *>(dev_buf);
    float *pos = (float *)p;      p += align256((N + 1) * 3 * sizeof(float));
    float *mass = (float *)p;     p += align256((N + 1) * sizeof(float));
    int *labels = (int *)p;       p += align256((N + 1) * sizeof(int));
    int *pgroup = (int *)p;       p += align256((N + 1) * sizeof(int));
    int *glabel = (int *)p;       p += align256(((size_t)cap + 1) * sizeof(int));
    int *gsize = (int *)p;        p += align256(((size_t)cap + 1) * sizeof(int));
    float *gmass = (float *)p;    p += align256(((size_t)cap + 1) * sizeof(float));
    float *gcom = (float *)p;     p += align256(((size_t)cap + 1) * 3 * sizeof(float));
    void *ws = p;
    cudaStream_t in = h->in_stream, run = h->run_stream;
    // Anything enqueued below is waited for by fof_host_wait, also after an error in the middle: the slot is
    // busy from the first copy on.
    sl.busy = true;
    sl.cap = -1;  // "the groups were not enqueued"
    if (N) CK(cudaMemcpyAsync(pos, pos_host, N * 3 * sizeof(float), cudaMemcpyHostToDevice, in), "H2D pos");
    if (N && mass_host) CK(cudaMemcpyAsync(mass, mass_host, N * sizeof(float), cudaMemcpyHostToDevice, in), "H2D mass");
    CK(cudaEventRecord(sl.ev_in, in), "cudaEventRecord");
    CK(cudaStreamWaitEvent(run, sl.ev_in, 0), "cudaStreamWaitEvent");
    int rc = fof_link(h, pos, labels, ws, run);
    if (rc != FOF_OK) return rc;
    CK(cudaEventRecord(sl.ev_linked, run), "cudaEventRecord");
    CK(cudaStreamWaitEvent(sl.out, sl.ev_linked, 0), "cudaStreamWaitEvent");
    if (N) CK(cudaMemcpyAsync(labels_host, labels, N * sizeof(int), cudaMemcpyDeviceToHost, sl.out), "D2H labels");
    rc = groups_enqueue(h, pos, mass_host ? mass : nullptr, labels, ws, glabel, gsize, gmass, gcom,
                        particle_group_host ? pgroup : nullptr, cap, run);
    if (rc != FOF_OK) return rc;
    // K and the error bits follow the labels on the slot's own copy stream: `run` never waits for a copy
    CK(cudaEventRecord(sl.ev_groups, run), "cudaEventRecord");
    CK(cudaStreamWaitEvent(sl.out, sl.ev_groups, 0), "cudaStreamWaitEvent");
    CK(cudaMemcpyAsync(sl.ctrl_pin, at<Ctrl>(ws, h->off_ctrl), sizeof(Ctrl), cudaMemcpyDeviceToHost, sl.out), "copy ctrl");
    CK(cudaEventRecord(sl.ev_ctrl, sl.out), "cudaEventRecord");
    if (N && particle_group_host)
        CK(cudaMemcpyAsync(particle_group_host, pgroup, N * sizeof(int), cudaMemcpyDeviceToHost, sl.out),
           "D2H particle_group");
    sl.cap = cap;
    sl.group_label_host = group_label_host; sl.group_size_host = group_size_host;
    sl.group_mass_host = group_mass_host;   sl.group_com_host = group_com_host;
    sl.glabel = glabel; sl.gsize = gsize; sl.gmass = gmass; sl.gcom = gcom;
    return FOF_OK;
}

int fof_host_wait(fof_handle *h, int32_t slot, int64_t *K_host)
{
    if (!h || slot < 0 || slot > 1 || !K_host) return FOF_ERR_INVALID_ARG;
    if (!h->in_stream || !h->slot[slot].busy) return FOF_ERR_STATE;
    fof_handle::HostSlot &sl = h->slot[slot];
    *K_host = 0;
    sl.busy = false;
    if (sl.cap < 0) {  // the submit failed half way: drain what it enqueued
        (void)cudaStreamSynchronize(h->in_stream);
        (void)cudaStreamSynchronize(h->run_stream);
        (void)cudaStreamSynchronize(sl.out);
        return FOF_ERR_STATE;
    }
    int rc = FOF_OK;
    cudaError_t e = cudaEventSynchronize(sl.ev_ctrl);  // K and the error bits are in ctrl_pin now
    if (e == cudaSuccess) {
        const long long K = sl.ctrl_pin->K;
        *K_host = (int64_t)K;
        if (K > sl.cap) rc = FOF_ERR_CAPACITY;
        else if (K > 0) {
            const size_t k = (size_t)K;
            e = cudaMemcpyAsync(sl.group_label_host, sl.glabel, k * sizeof(int), cudaMemcpyDeviceToHost, sl.out);
            if (e == cudaSuccess)
                e = cudaMemcpyAsync(sl.group_size_host, sl.gsize, k * sizeof(int), cudaMemcpyDeviceToHost, sl.out);
            if (e == cudaSuccess)
                e = cudaMemcpyAsync(sl.group_mass_host, sl.gmass, k * sizeof(float), cudaMemcpyDeviceToHost, sl.out);
            if (e == cudaSuccess)
                e = cudaMemcpyAsync(sl.group_com_host, sl.gcom, k * 3 * sizeof(float), cudaMemcpyDeviceToHost, sl.out);
        }
    }
    const cudaError_t e2 = cudaStreamSynchronize(sl.out);  // always: the caller's buffers are free after this call
    if (e != cudaSuccess) return cuda_fail(h, e, "fof_host_wait");
    if (e2 != cudaSuccess) return cuda_fail(h, e2, "fof_host_wait");
    if (rc != FOF_OK) return rc;
    if (sl.ctrl_pin->error & 1u) return FOF_ERR_NONFINITE;
    return FOF_OK;
}

int fof_status(fof_handle *h, void *ws, void *stream)
{
    if (!h || !ws) return FOF_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    Ctrl c;
    CK(cudaMemcpyAsync(&c, at<Ctrl>(ws, h->off_ctrl), sizeof(Ctrl), cudaMemcpyDeviceToHost, s), "copy ctrl");
    CK(cudaStreamSynchronize(s), "sync");
    if (c.error & 1u) return FOF_ERR_NONFINITE;
    return FOF_OK;
}

const char *fof_error_string(int code)
{
    switch (code) {
    case FOF_OK: return "ok";
    case FOF_ERR_INVALID_ARG: return "invalid argument";
    case FOF_ERR_UNSUPPORTED: return "unsupported: fewer than 3 cells of side >= b per axis";
    case FOF_ERR_CUDA: return "CUDA runtime error";
    case FOF_ERR_NONFINITE: return "non-finite position";
    case FOF_ERR_CAPACITY: return "more groups than capacity";
    case FOF_ERR_STATE: return "call order violated";
    default: return "unknown error";
    }
}

const char *fof_last_cuda_error(const fof_handle *h) { return h ? h->cuda_err : ""; }

}  // extern "C"
