// kernels_groups.cu — H6 sizes, H7 compaction, H8 masses and periodic centres of mass.
// PAPER.md:93-95 (§2 step vi), PAPER.md:172 ("accumulates particle counts per halo via a parallel
// histogram"), PAPER.md:227 (Alg. 2 "Compaction"), PAPER.md:259 (Eq. 4, halo position = mean of
// member positions; made periodic per DESIGN.md R11), PAPER.md:263/369 (minimum particle cut).
//
// All three passes are latency-bound gathers / atomics over N particles, so every thread takes
// four consecutive particles and issues their loads together (128-bit where the pointers allow).
#include "fof_internal.cuh"

namespace fof {

#ifndef FOF_GROUP_PER
#define FOF_GROUP_PER 4
#endif
constexpr int kPer = FOF_GROUP_PER;  // particles per thread in the streaming passes (multiple of 4)

template <bool VEC>
__device__ __forceinline__ void load_per(const int *__restrict__ p, int64_t i, int64_t N, int v[kPer], int fill)
{
    if (VEC && i + kPer <= N) {
#pragma unroll
        for (int q = 0; q < kPer / 4; ++q) {
            const int4 t = __ldg(reinterpret_cast<const int4 *>(p + i + 4 * q));
            v[4 * q] = t.x; v[4 * q + 1] = t.y; v[4 * q + 2] = t.z; v[4 * q + 3] = t.w;
        }
    } else {
#pragma unroll
        for (int k = 0; k < kPer; ++k) v[k] = (i + k < N) ? __ldg(p + i + k) : fill;
    }
}

// H6: cnt[g] = number of members of group g other than its canonical particle (labels[i] != i).
// Singletons (most of the background) issue no atomic at all.
template <bool VEC>
__global__ void __launch_bounds__(kBlock) group_count_kernel(const int *__restrict__ labels, int64_t N,
                                                             int *__restrict__ cnt, unsigned long long *state,
                                                             int64_t state_items, Ctrl *ctrl)
{
    // also clears what group_compact_kernel (the next launch) needs: its ticket, K and scan state
    const int64_t tid = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (tid == 0) { ctrl->gscan_ticket = 0u; ctrl->K = 0; }
    for (int64_t k = tid; k < state_items; k += (int64_t)gridDim.x * kBlock) state[k] = 0ull;
    const int64_t i = tid * kPer;
    if (i >= N) return;
    int l[kPer];
    load_per<VEC>(labels, i, N, l, -1);
#pragma unroll
    for (int k = 0; k < kPer; ++k)
        if (l[k] >= 0 && l[k] != (int)(i + k)) atomicAdd(cnt + l[k], 1);
}

// H7: a canonical particle i (labels[i] == i) heads a kept group iff cnt[i] + 1 >= N_min; the
// exclusive scan of that flag over i is the compact id, ascending in the canonical label.  Single
// pass with decoupled look-back: state[tile] = (flag << 32) | value, flag 1 = tile aggregate,
// 2 = inclusive prefix; tiles are handed out by an atomic ticket, so a tile only ever waits on
// tiles that already started.  In place: the entry of a kept canonical particle becomes
// -1 - gid; every other entry stays >= 0 (a count), which H8 reads as "dropped".
// For N_min >= 2 the labels are not read at all: cnt[i] > 0 already says that i is canonical.
__device__ __forceinline__ unsigned int lookback_g(unsigned long long *state, unsigned int tile,
                                                   unsigned int aggregate, int lane)
{
    unsigned int exclusive = 0;
    int64_t idx = (int64_t)tile - 1;
    while (true) {
        int64_t j = idx - lane;
        unsigned long long v = (2ull << 32);
        if (j >= 0) {
            do { v = ld_relaxed_u64(state + j); } while ((v >> 32) == 0);
        }
        unsigned int flag = (unsigned int)(v >> 32), val = (unsigned int)v;
        unsigned int full = __ballot_sync(0xffffffffu, flag == 2);
        int stop = full ? __ffs(full) - 1 : 31;
        unsigned int part = (lane <= stop) ? val : 0;
        for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
        exclusive += part;
        if (full) break;
        idx -= 32;
    }
    if (lane == 0) st_relaxed_u64(state + tile, (2ull << 32) | (unsigned long long)(exclusive + aggregate));
    return exclusive;
}

__global__ void __launch_bounds__(kBlock) group_compact_kernel(const int *__restrict__ labels, int64_t N, int N_min,
                                                               int *cnt_to_gid, int64_t cap,
                                                               int *__restrict__ group_label,
                                                               int *__restrict__ group_size, double *__restrict__ acc,
                                                               unsigned long long *state, Ctrl *ctrl,
                                                               unsigned int last_tile)
{
    __shared__ unsigned int s_tile, s_prefix;
    __shared__ unsigned int s_warp[kBlock / 32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(&ctrl->gscan_ticket, 1u);
    __syncthreads();
    const unsigned int tile = s_tile;
    const int64_t base = (int64_t)tile * kScanTile + (int64_t)tid * kScanItems;

    int c[kScanItems];
    if (base + kScanItems <= N) {  // cnt is a workspace array: 16-byte aligned
#pragma unroll
        for (int q = 0; q < kScanItems / 4; ++q) {
            const int4 a = *reinterpret_cast<const int4 *>(cnt_to_gid + base + 4 * q);
            c[4 * q] = a.x; c[4 * q + 1] = a.y; c[4 * q + 2] = a.z; c[4 * q + 3] = a.w;
        }
    } else {
#pragma unroll
        for (int k = 0; k < kScanItems; ++k) c[k] = (base + k < N) ? cnt_to_gid[base + k] : -1;
    }
    unsigned int keep = 0;  // bit k: item k is the canonical particle of a kept group
    if (N_min >= 2) {
#pragma unroll
        for (int k = 0; k < kScanItems; ++k)
            if (c[k] + 1 >= N_min) keep |= 1u << k;
    } else {
#pragma unroll
        for (int k = 0; k < kScanItems; ++k)
            if (base + k < N && labels[base + k] == (int)(base + k)) keep |= 1u << k;
    }
    const unsigned int sum = __popc(keep);
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
            unsigned int ex = lookback_g(state, tile, total, lane);
            if (lane == 0) s_prefix = ex;
        }
    }
    __syncthreads();
    unsigned int k_out = s_prefix + warp_off + (incl - sum);
    if (tile == last_tile && tid == kBlock - 1) ctrl->K = (long long)s_prefix + total;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        if (!(keep & (1u << k))) continue;
        const int64_t i = base + k;
        const int gid = (int)k_out++;
        cnt_to_gid[i] = -1 - gid;
        if (gid < cap) {
            group_label[gid] = (int)i;
            group_size[gid] = c[k] + 1;
            double2 *a2 = reinterpret_cast<double2 *>(acc + 4 * (int64_t)gid);
            a2[0] = make_double2(0.0, 0.0);
            a2[1] = make_double2(0.0, 0.0);
        }
    }
}

// H8 accumulate: for every member of a kept group, delta = min-image(w_i - r) in double with
// r = wrapped position of the canonical particle; acc[g] += (m dx, m dy, m dz, m).
// The pass is bound by the L2 atomic rate (three or four float64 atomics per member), so groups of
// fewer than kFloatAccMax members use ONE 128-bit float32 atomic per member instead (the same
// 32-byte slot read as a float4): with deltas of at most L/2 and < 4096 terms the float32 sums stay
// ~1e-3 ulp(L) per member away from the float64 ones, far inside the 1e-5 L tolerance; larger groups
// (a percolating component) keep float64.
constexpr int kFloatAccMax = 4096;
__device__ __forceinline__ double min_image_d(double d, double L, double h)
{
    if (d > h) d -= L;
    else if (d < -h) d += L;
    return d;
}

template <bool VEC>
__global__ void __launch_bounds__(kBlock) group_reduce_kernel(const float *__restrict__ pos,
                                                              const float *__restrict__ mass,
                                                              const int *__restrict__ labels, int64_t N, Grid g,
                                                              const int *__restrict__ gid_of, int64_t cap,
                                                              const int *__restrict__ group_size, double *acc,
                                                              int *__restrict__ particle_group)
{
    const int64_t i0 = ((int64_t)blockIdx.x * kBlock + threadIdx.x) * kPer;
    if (i0 >= N) return;
    int l[kPer], gid[kPer];
    load_per<VEC>(labels, i0, N, l, -1);
#pragma unroll
    for (int k = 0; k < kPer; ++k) gid[k] = l[k] >= 0 ? -1 - __ldg(gid_of + l[k]) : -1;  // < 0: dropped
    if (particle_group) {
        if (VEC && i0 + kPer <= N) {
#pragma unroll
            for (int q = 0; q < kPer / 4; ++q)
                *reinterpret_cast<int4 *>(particle_group + i0 + 4 * q) =
                    make_int4(max(gid[4 * q], -1), max(gid[4 * q + 1], -1), max(gid[4 * q + 2], -1),
                              max(gid[4 * q + 3], -1));
        } else {
#pragma unroll
            for (int k = 0; k < kPer; ++k)
                if (i0 + k < N) particle_group[i0 + k] = max(gid[k], -1);
        }
    }
    const double L = (double)g.L, h = 0.5 * (double)g.L;
    // Consecutive particles of one group (snapshots keep neighbours together: here the members of a halo are
    // contiguous in the input) are summed in registers first: one atomic per run instead of one per member.
    double run[4] = {0.0, 0.0, 0.0, 0.0};
    int run_gid = -1;
    auto flush = [&]() {
        if (run_gid < 0) return;
        double *dst = acc + 4 * (int64_t)run_gid;
        if (__ldg(group_size + run_gid) < kFloatAccMax) {
            if (run[0] != 0.0 || run[1] != 0.0 || run[2] != 0.0 || run[3] != 0.0)
                atomicAdd(reinterpret_cast<float4 *>(dst), make_float4((float)run[0], (float)run[1], (float)run[2], (float)run[3]));
        } else {
            if (run[0] != 0.0) atomicAdd(dst + 0, run[0]);
            if (run[1] != 0.0) atomicAdd(dst + 1, run[1]);
            if (run[2] != 0.0) atomicAdd(dst + 2, run[2]);
            if (run[3] != 0.0) atomicAdd(dst + 3, run[3]);
        }
        run[0] = run[1] = run[2] = run[3] = 0.0;
    };
#pragma unroll
    for (int k = 0; k < kPer; ++k) {
        if (gid[k] < 0 || gid[k] >= cap) continue;
        const int64_t i = i0 + k;
        if (gid[k] != run_gid) { flush(); run_gid = gid[k]; }
        const double m = mass ? (double)__ldg(mass + i) : 1.0;
        if (l[k] != (int)i) {  // the canonical particle itself has delta = 0
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const float wi = wrap1(__ldg(pos + 3 * i + a), g.L);
                const float wr = wrap1(__ldg(pos + 3 * (int64_t)l[k] + a), g.L);
                run[a] += m * min_image_d((double)wi - (double)wr, L, h);
            }
        }
        if (mass) run[3] += m;
    }
    flush();
}

// H8 finish: one thread per kept group.
__global__ void __launch_bounds__(kBlock) group_finish_kernel(const float *__restrict__ pos,
                                                              const int *__restrict__ group_label,
                                                              const int *__restrict__ group_size,
                                                              const double *__restrict__ acc, bool has_mass, Grid g,
                                                              int64_t cap, const Ctrl *ctrl,
                                                              float *__restrict__ group_mass,
                                                              float *__restrict__ group_com)
{
    const int64_t k = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    long long K = ctrl->K;
    if (K > cap) K = cap;
    if (k >= K) return;
    const int l = group_label[k];
    double sum[4];
    if (group_size[k] < kFloatAccMax) {  // float32 slot (see group_reduce_kernel)
        const float4 f = *reinterpret_cast<const float4 *>(acc + 4 * k);
        sum[0] = f.x; sum[1] = f.y; sum[2] = f.z; sum[3] = f.w;
    } else {
        sum[0] = acc[4 * k]; sum[1] = acc[4 * k + 1]; sum[2] = acc[4 * k + 2]; sum[3] = acc[4 * k + 3];
    }
    const double M = has_mass ? sum[3] : (double)group_size[k];
    const double L = (double)g.L;
    group_mass[k] = (float)M;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const float wr = wrap1(pos[3 * (int64_t)l + a], g.L);
        double c = (double)wr + sum[a] / M;
        if (c < 0.0) c += L;
        if (c >= L) c -= L;
        float cf = (float)c;
        if (cf >= g.L) cf = 0.0f;
        group_com[3 * k + a] = cf;
    }
}

static inline unsigned int blocks_for(int64_t n, int per_block) { return (unsigned int)((n + per_block - 1) / per_block); }
static inline bool aligned16(const void *p) { return ((uintptr_t)p & 15) == 0; }

cudaError_t launch_group_count(const int *labels, int64_t N, int *cnt, unsigned long long *state,
                               int64_t state_items, Ctrl *ctrl, cudaStream_t s)
{
    const unsigned int grid = N > 0 ? blocks_for(N, kBlock * kPer) : 1u;
    if (aligned16(labels)) group_count_kernel<true><<<grid, kBlock, 0, s>>>(labels, N, cnt, state, state_items, ctrl);
    else group_count_kernel<false><<<grid, kBlock, 0, s>>>(labels, N, cnt, state, state_items, ctrl);
    return cudaGetLastError();
}

cudaError_t launch_group_compact(const int *labels, int64_t N, int N_min, int *cnt_to_gid, int64_t cap,
                                 int *group_label, int *group_size, double *acc, unsigned long long *state,
                                 Ctrl *ctrl, int64_t tiles, cudaStream_t s)
{
    if (N > 0)
        group_compact_kernel<<<(unsigned int)tiles, kBlock, 0, s>>>(labels, N, N_min, cnt_to_gid, cap, group_label,
                                                                    group_size, acc, state, ctrl,
                                                                    (unsigned int)(tiles - 1));
    return cudaGetLastError();
}

cudaError_t launch_group_reduce(const float *pos, const float *mass, const int *labels, int64_t N, Grid g,
                                const int *gid, int64_t cap, const int *group_size, double *acc, int *particle_group,
                                cudaStream_t s)
{
    if (N <= 0) return cudaSuccess;
    const unsigned int grid = blocks_for(N, kBlock * kPer);
    if (aligned16(labels) && aligned16(particle_group))
        group_reduce_kernel<true><<<grid, kBlock, 0, s>>>(pos, mass, labels, N, g, gid, cap, group_size, acc, particle_group);
    else
        group_reduce_kernel<false><<<grid, kBlock, 0, s>>>(pos, mass, labels, N, g, gid, cap, group_size, acc, particle_group);
    return cudaGetLastError();
}

cudaError_t launch_group_finish(const float *pos, const int *group_label, const int *group_size,
                                const double *acc, bool has_mass, Grid g, int64_t cap, const Ctrl *ctrl,
                                float *group_mass, float *group_com, cudaStream_t s)
{
    if (cap > 0)
        group_finish_kernel<<<blocks_for(cap, kBlock), kBlock, 0, s>>>(pos, group_label, group_size, acc, has_mass,
                                                                      g, cap, ctrl, group_mass, group_com);
    return cudaGetLastError();
}

}  // namespace fof
