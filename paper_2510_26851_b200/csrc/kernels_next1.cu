// kernels_next1.cu — halo decoration sigma and frozen-assignment backward.
// PAPER.md:255-261 (section 3.1 "Frozen Assignment", Eq. 4: dX^h/dtheta = (1/N) sum dx_i/dtheta) and
// PAPER.md:283-290 (section 3.1.1 "Decorated Frozen Assignment", Eq. 5; decoration = particle
// standard deviation sigma).  Readings R23 / R24 of DESIGN.md: sigma_g = sqrt(sum m |delta|^2 / M),
// delta = minimum-image displacement from the periodic centre of mass;
// dL/dx_i = (m_i / M_g) (dL/dX_g + dL/dsigma_g delta_i / sigma_g), 0 for dropped particles.
// Both are single streaming passes over the particles, downstream of fof_groups (they read its
// particle_group, group_mass and group_com outputs); arithmetic in float64, outputs float32.
#include "fof_internal.cuh"

namespace fof {

__device__ __forceinline__ void delta_from_com(const float *__restrict__ pos, int64_t i, const float *__restrict__ com,
                                               int k, const Grid &g, double d[3])
{
    const double L = (double)g.L, h = 0.5 * (double)g.L;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        double v = (double)wrap1(__ldg(pos + 3 * i + a), g.L) - (double)__ldg(com + 3 * (int64_t)k + a);
        if (v > h) v -= L;
        else if (v < -h) v += L;
        d[a] = v;
    }
}

// four consecutive particles per thread: one 128-bit load of their group ids
template <bool VEC>
__device__ __forceinline__ void load_ids4(const int *__restrict__ pg, int64_t i0, int64_t N, int k[4])
{
    if (VEC && i0 + 3 < N) {
        const int4 t = __ldg(reinterpret_cast<const int4 *>(pg + i0));
        k[0] = t.x; k[1] = t.y; k[2] = t.z; k[3] = t.w;
    } else {
#pragma unroll
        for (int q = 0; q < 4; ++q) k[q] = (i0 + q < N) ? __ldg(pg + i0 + q) : -1;
    }
}

template <bool VEC>
__global__ void __launch_bounds__(kBlock) sigma_accum_kernel(const float *__restrict__ pos,
                                                             const float *__restrict__ mass,
                                                             const int *__restrict__ particle_group, int64_t N, Grid g,
                                                             const float *__restrict__ group_com, int64_t K,
                                                             double *acc)
{
    const int64_t i0 = ((int64_t)blockIdx.x * kBlock + threadIdx.x) * 4;
    if (i0 >= N) return;
    int k[4];
    load_ids4<VEC>(particle_group, i0, N, k);
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        if (k[q] < 0 || k[q] >= K) continue;
        double d[3];
        delta_from_com(pos, i0 + q, group_com, k[q], g, d);
        const double m = mass ? (double)__ldg(mass + i0 + q) : 1.0;
        atomicAdd(acc + k[q], m * (d[0] * d[0] + d[1] * d[1] + d[2] * d[2]));
    }
}

__global__ void __launch_bounds__(kBlock) sigma_finish_kernel(const double *__restrict__ acc,
                                                              const float *__restrict__ group_mass, int64_t K,
                                                              float *__restrict__ group_sigma)
{
    const int64_t k = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (k >= K) return;
    const double M = (double)group_mass[k];
    group_sigma[k] = M > 0.0 ? (float)sqrt(acc[k] / M) : 0.0f;
}

template <bool VEC>
__global__ void __launch_bounds__(kBlock) groups_backward_kernel(
    const float *__restrict__ pos, const float *__restrict__ mass, const int *__restrict__ particle_group, int64_t N,
    Grid g, const float *__restrict__ group_mass, const float *__restrict__ group_com,
    const float *__restrict__ group_sigma, const float *__restrict__ grad_com, const float *__restrict__ grad_sigma,
    int64_t K, float *__restrict__ grad_pos)
{
    const int64_t i0 = ((int64_t)blockIdx.x * kBlock + threadIdx.x) * 4;
    if (i0 >= N) return;
    int k[4];
    load_ids4<VEC>(particle_group, i0, N, k);
    float out[12];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        double o[3] = {0.0, 0.0, 0.0};
        if (k[q] >= 0 && k[q] < K) {
            const int64_t i = i0 + q;
            const double m = mass ? (double)__ldg(mass + i) : 1.0;
            const double wgt = m / (double)__ldg(group_mass + k[q]);
            if (grad_com) {
#pragma unroll
                for (int a = 0; a < 3; ++a) o[a] = wgt * (double)__ldg(grad_com + 3 * (int64_t)k[q] + a);
            }
            if (grad_sigma) {
                const double s = (double)__ldg(group_sigma + k[q]);
                if (s > 0.0) {
                    double d[3];
                    delta_from_com(pos, i, group_com, k[q], g, d);
                    const double c = (double)__ldg(grad_sigma + k[q]) * wgt / s;
#pragma unroll
                    for (int a = 0; a < 3; ++a) o[a] += c * d[a];
                }
            }
        }
#pragma unroll
        for (int a = 0; a < 3; ++a) out[3 * q + a] = (float)o[a];
    }
    if (VEC && i0 + 3 < N) {  // 48 contiguous bytes: three 128-bit stores
        float4 *dst = reinterpret_cast<float4 *>(grad_pos + 3 * i0);
        dst[0] = make_float4(out[0], out[1], out[2], out[3]);
        dst[1] = make_float4(out[4], out[5], out[6], out[7]);
        dst[2] = make_float4(out[8], out[9], out[10], out[11]);
    } else {
#pragma unroll
        for (int q = 0; q < 4; ++q)
            if (i0 + q < N) {
#pragma unroll
                for (int a = 0; a < 3; ++a) grad_pos[3 * (i0 + q) + a] = out[3 * q + a];
            }
    }
}

static inline unsigned int blocks_for(int64_t n, int per_block) { return (unsigned int)((n + per_block - 1) / per_block); }

cudaError_t launch_group_sigma(const float *pos, const float *mass, const int *particle_group, int64_t N, Grid g,
                               const float *group_mass, const float *group_com, int64_t K, double *acc,
                               float *group_sigma, cudaStream_t s)
{
    if (K <= 0) return cudaSuccess;
    cudaError_t e = cudaMemsetAsync(acc, 0, (size_t)K * sizeof(double), s);
    if (e != cudaSuccess) return e;
    if (N > 0) {
        const unsigned int grid = blocks_for(N, kBlock * 4);
        if (((uintptr_t)particle_group & 15) == 0)
            sigma_accum_kernel<true><<<grid, kBlock, 0, s>>>(pos, mass, particle_group, N, g, group_com, K, acc);
        else
            sigma_accum_kernel<false><<<grid, kBlock, 0, s>>>(pos, mass, particle_group, N, g, group_com, K, acc);
    }
    sigma_finish_kernel<<<blocks_for(K, kBlock), kBlock, 0, s>>>(acc, group_mass, K, group_sigma);
    return cudaGetLastError();
}

cudaError_t launch_groups_backward(const float *pos, const float *mass, const int *particle_group, int64_t N, Grid g,
                                   const float *group_mass, const float *group_com, const float *group_sigma,
                                   const float *grad_com, const float *grad_sigma, int64_t K, float *grad_pos,
                                   cudaStream_t s)
{
    if (N > 0) {
        const unsigned int grid = blocks_for(N, kBlock * 4);
        if ((((uintptr_t)particle_group | (uintptr_t)grad_pos) & 15) == 0)
            groups_backward_kernel<true><<<grid, kBlock, 0, s>>>(pos, mass, particle_group, N, g, group_mass, group_com,
                                                                 group_sigma, grad_com, grad_sigma, K, grad_pos);
        else
            groups_backward_kernel<false><<<grid, kBlock, 0, s>>>(pos, mass, particle_group, N, g, group_mass, group_com,
                                                                  group_sigma, grad_com, grad_sigma, K, grad_pos);
    }
    return cudaGetLastError();
}

}  // namespace fof
