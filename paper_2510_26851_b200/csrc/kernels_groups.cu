// kernels_groups.cu — H6 sizes, H7 compaction, H8 masses and periodic centres of mass.
// PAPER.md:93-95 (§2 step vi), PAPER.md:172 ("accumulates particle counts per halo via a parallel
// histogram"), PAPER.md:227 (Alg. 2 "Compaction"), PAPER.md:259 (Eq. 4, halo position = mean of
// member positions; made periodic per DESIGN.md R11), PAPER.md:263/369 (minimum particle cut).
#include "fof_internal.cuh"

namespace fof {

// H6: cnt[g] = number of members of group g other than its canonical particle (labels[i] != i).
// Singletons (most of the background) issue no atomic at all.
__global__ void __launch_bounds__(kBlock) group_count_kernel(const int *__restrict__ labels, int64_t N,
                                                             int *__restrict__ cnt)
{
    const int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (i >= N) return;
    const int l = labels[i];
    if (l != (int)i) atomicAdd(cnt + l, 1);
}

// H7: kept[i] = (labels[i] == i && cnt[i] + 1 >= N_min); exclusive scan of kept over i gives the
// compact id, ascending in the canonical label.  Same single-pass look-back scan as the cell scan.
// In place: cnt[i] becomes gid[i] (compact id of the group whose canonical particle is i, else -1).
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

    int sz[kScanItems];
    unsigned int keep = 0;  // bit k: item k is the canonical particle of a kept group
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        const int64_t i = base + k;
        sz[k] = 0;
        if (i < N) {
            const int c = cnt_to_gid[i];
            if (labels[i] == (int)i && c + 1 >= N_min) { keep |= 1u << k; sz[k] = c + 1; }
        }
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
        const int64_t i = base + k;
        if (i >= N) break;
        int gid = -1;
        if (keep & (1u << k)) {
            gid = (int)k_out++;
            if (gid < cap) {
                group_label[gid] = (int)i;
                group_size[gid] = sz[k];
                acc[4 * (int64_t)gid + 0] = 0.0;
                acc[4 * (int64_t)gid + 1] = 0.0;
                acc[4 * (int64_t)gid + 2] = 0.0;
                acc[4 * (int64_t)gid + 3] = 0.0;
            }
        }
        cnt_to_gid[i] = gid;
    }
}

// H8 accumulate: for every member of a kept group, delta = min-image(w_i - r) in double with
// r = wrapped position of the canonical particle; acc[g] += (m dx, m dy, m dz, m).
__device__ __forceinline__ double min_image_d(double d, double L, double h)
{
    if (d > h) d -= L;
    else if (d < -h) d += L;
    return d;
}

__global__ void __launch_bounds__(kBlock) group_reduce_kernel(const float *__restrict__ pos,
                                                              const float *__restrict__ mass,
                                                              const int *__restrict__ labels, int64_t N, Grid g,
                                                              const int *__restrict__ gid_of, int64_t cap,
                                                              double *acc, int *__restrict__ particle_group)
{
    const int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (i >= N) return;
    const int l = labels[i];
    const int gid = gid_of[l];
    if (particle_group) particle_group[i] = gid;
    if (gid < 0 || gid >= cap) return;
    const double L = (double)g.L, h = 0.5 * (double)g.L;
    const double m = mass ? (double)mass[i] : 1.0;
    double d[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const float wi = wrap1(pos[3 * i + a], g.L);
        const float wr = wrap1(pos[3 * (int64_t)l + a], g.L);
        d[a] = min_image_d((double)wi - (double)wr, L, h);
    }
    double *dst = acc + 4 * (int64_t)gid;
    if (l != (int)i) {  // the canonical particle itself has delta = 0
        atomicAdd(dst + 0, m * d[0]);
        atomicAdd(dst + 1, m * d[1]);
        atomicAdd(dst + 2, m * d[2]);
    }
    if (mass) atomicAdd(dst + 3, m);
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
    const double M = has_mass ? acc[4 * k + 3] : (double)group_size[k];
    const double L = (double)g.L;
    group_mass[k] = (float)M;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const float wr = wrap1(pos[3 * (int64_t)l + a], g.L);
        double c = (double)wr + acc[4 * k + a] / M;
        if (c < 0.0) c += L;
        if (c >= L) c -= L;
        float cf = (float)c;
        if (cf >= g.L) cf = 0.0f;
        group_com[3 * k + a] = cf;
    }
}

static inline unsigned int blocks_for(int64_t n, int per_block) { return (unsigned int)((n + per_block - 1) / per_block); }

cudaError_t launch_group_count(const int *labels, int64_t N, int *cnt, cudaStream_t s)
{
    if (N > 0) group_count_kernel<<<blocks_for(N, kBlock), kBlock, 0, s>>>(labels, N, cnt);
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
                                const int *gid, int64_t cap, double *acc, int *particle_group, cudaStream_t s)
{
    if (N > 0)
        group_reduce_kernel<<<blocks_for(N, kBlock), kBlock, 0, s>>>(pos, mass, labels, N, g, gid, cap, acc,
                                                                     particle_group);
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
