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

// offsets[k] = sum of group_size[0..k), offsets[K] = number of members; cursor[k] = 0.  One CTA.
__global__ void __launch_bounds__(1024) sub_offsets_kernel(const int *__restrict__ group_size, int64_t K,
                                                           unsigned int *__restrict__ offsets,
                                                           unsigned int *__restrict__ cursor)
{
    __shared__ unsigned int s_warp[32];
    __shared__ unsigned int s_carry;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) s_carry = 0u;
    __syncthreads();
    for (int64_t base = 0; base < K; base += 1024) {
        const int64_t k = base + threadIdx.x;
        const unsigned int v = k < K ? (unsigned int)group_size[k] : 0u;
        unsigned int incl = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        unsigned int off = s_carry, tot = 0;
        for (int w = 0; w < 32; ++w) {
            const unsigned int t = s_warp[w];
            if (w < warp) off += t;
            tot += t;
        }
        if (k < K) { offsets[k] = off + incl - v; cursor[k] = 0u; }
        __syncthreads();
        if (threadIdx.x == 0) s_carry += tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) offsets[K] = s_carry;
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

__device__ __forceinline__ bool linked6(const float *a, const float *b, const Sub6 &q)
{
    const float dx = min_image(__fsub_rn(a[0], b[0]), q.L, q.h), dy = min_image(__fsub_rn(a[1], b[1]), q.L, q.h),
                dz = min_image(__fsub_rn(a[2], b[2]), q.L, q.h);
    const float ux = __fsub_rn(a[3], b[3]), uy = __fsub_rn(a[4], b[4]), uz = __fsub_rn(a[5], b[5]);
    const float dx2 = __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
    const float dv2 = __fadd_rn(__fadd_rn(__fmul_rn(ux, ux), __fmul_rn(uy, uy)), __fmul_rn(uz, uz));
    return __fadd_rn(__fmul_rn(dx2, q.rx), __fmul_rn(dv2, q.rv)) <= q.ell2;
}

constexpr int kSubWarps = kBlock / 32;

// One warp per tile of 32 member slots; the tile meets itself and every earlier tile; a pair is
// taken by its later slot.  Two launches share the halos by size: WIDE = false, one warp per halo of
// at most kSubSmall members (eight halos per CTA: a typical halo has two tiles); WIDE = true, one CTA
// per larger halo, its warps striding over the tiles.
constexpr int kSubSmall = 256;

template <bool WIDE>
__global__ void __launch_bounds__(kBlock) subhalo_link_kernel(const float *__restrict__ pos,
                                                              const float *__restrict__ vel, int64_t K, Sub6 q,
                                                              const unsigned int *__restrict__ offsets,
                                                              const int *__restrict__ members, unsigned int *sub_rel,
                                                              Ctrl *ctrl)
{
    __shared__ float s_j[kSubWarps][32][6];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned int nedges = 0;
    const int64_t k0 = WIDE ? (int64_t)blockIdx.x : (int64_t)blockIdx.x * kSubWarps + warp;
    const int64_t kstep = WIDE ? (int64_t)gridDim.x : (int64_t)gridDim.x * kSubWarps;
    for (int64_t k = k0; k < K; k += kstep) {
        const int off = (int)offsets[k], M = (int)offsets[k + 1] - off;
        if ((M > kSubSmall) != WIDE) continue;
        const int tiles = (M + 31) >> 5;
        for (int it = WIDE ? warp : 0; it < tiles; it += WIDE ? kSubWarps : 1) {
            const int myslot = off + it * 32 + lane;
            const bool valid = it * 32 + lane < M;
            float me[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
            if (valid) {
                const int64_t i = members[myslot];
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    me[a] = wrap1(__ldg(pos + 3 * i + a), q.L);
                    me[3 + a] = __ldg(vel + 3 * i + a);
                }
            }
            for (int jt = 0; jt <= it; ++jt) {
                __syncwarp();
                const int jslot0 = off + jt * 32;
                const int cnt = min(32, M - jt * 32);
                if (jt == it) {
#pragma unroll
                    for (int a = 0; a < 6; ++a) s_j[warp][lane][a] = me[a];
                } else {  // earlier tiles are full
                    const int64_t j = members[jslot0 + lane];
#pragma unroll
                    for (int a = 0; a < 3; ++a) {
                        s_j[warp][lane][a] = wrap1(__ldg(pos + 3 * j + a), q.L);
                        s_j[warp][lane][3 + a] = __ldg(vel + 3 * j + a);
                    }
                }
                __syncwarp();
                for (int c = 0; c < cnt; ++c) {
                    const int jslot = jslot0 + c;
                    if (valid && jslot < myslot && linked6(me, s_j[warp][c], q)) {
                        ++nedges;
                        const int pa = myslot - (int)sub_rel[myslot], pb = jslot - (int)sub_rel[jslot];
                        if (pa != pb) unite_rel(sub_rel, members, myslot, jslot);  // same parent: already one set
                    }
                }
            }
        }
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
    sub_offsets_kernel<<<1, 1024, 0, s>>>(group_size, K, offsets, cursor);
    sub_fill_kernel<<<(unsigned int)((N + kBlock - 1) / kBlock), kBlock, 0, s>>>(particle_group, N, K, offsets, cursor,
                                                                                members, sub_rel, sub_labels);
    if (K > 0) {
        const int64_t cap = (int64_t)num_sms * 16;
        const unsigned int grid_small = (unsigned int)((K + kSubWarps - 1) / kSubWarps < cap ? (K + kSubWarps - 1) / kSubWarps : cap);
        const unsigned int grid_wide = (unsigned int)(K < cap ? K : cap);
        subhalo_link_kernel<false><<<grid_small, kBlock, 0, s>>>(pos, vel, K, q, offsets, members, sub_rel, ctrl);
        subhalo_link_kernel<true><<<grid_wide, kBlock, 0, s>>>(pos, vel, K, q, offsets, members, sub_rel, ctrl);
        sub_labels_kernel<<<(unsigned int)num_sms * 8, kBlock, 0, s>>>(sub_rel, members, offsets + K, sub_labels);
    }
    return cudaGetLastError();
}

}  // namespace fof
