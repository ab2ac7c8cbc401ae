// kernels_measure.cu — measurement aids (they compute nothing of the method): the ceilings that bench.py and
// DESIGN.md quote are measured on the box, not derived from a data sheet ("an FP32
// instruction-issue ceiling measured by a micro-benchmark on the box").
//   fof_measure_fp32_issue   non-FMA FP32 lane-operations per second (FADD + FMUL, the mix of the link predicate)
//   fof_measure_scatter      records per second of a copy whose 16-byte stores (or loads) are scattered inside
//                            windows of 2^k records: the floor of every reorder pass of H3
#include <math.h>

#include "fof_internal.cuh"

namespace fof {
namespace {

constexpr int kChains = 8;

// kChains independent chains of x <- (x * a) + b per thread, explicit _rn intrinsics so that nvcc cannot contract
// them into FMAs: 2 FP32 operations per chain step, all on the pipes the link predicate uses.
__global__ void __launch_bounds__(256) fp32_issue_kernel(float *out, int iters, float a, float b)
{
    float x[kChains];
#pragma unroll
    for (int k = 0; k < kChains; ++k) x[k] = (float)(threadIdx.x + k);
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < kChains; ++k) x[k] = __fadd_rn(__fmul_rn(x[k], a), b);
    }
    float s = 0.0f;
#pragma unroll
    for (int k = 0; k < kChains; ++k) s += x[k];
    if (s == 12345.678f) out[0] = s;  // never true: keeps the chains alive
}

// each thread moves 4 records, consecutive threads consecutive records; the scattered side is
// window base | ((index in window * odd) mod window)
template <bool SCATTER_STORE>
__global__ void __launch_bounds__(256) scramble_kernel(const float4 *__restrict__ in, float4 *__restrict__ out, int64_t n,
                                                       unsigned int wmask)
{
    const int64_t base = (int64_t)blockIdx.x * 1024 + threadIdx.x;
    float4 v[4];
    int64_t idx[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int64_t i = base + 256 * k;
        idx[k] = (i & ~(int64_t)wmask) | (int64_t)((((unsigned int)i & wmask) * 0x9E3779B1u) & wmask);
    }
    if (base + 768 >= n) return;
#pragma unroll
    for (int k = 0; k < 4; ++k) v[k] = in[SCATTER_STORE ? base + 256 * k : idx[k]];
#pragma unroll
    for (int k = 0; k < 4; ++k) out[SCATTER_STORE ? idx[k] : base + 256 * k] = v[k];
}

}  // namespace
}  // namespace fof

using namespace fof;

extern "C" {

int fof_measure_fp32_issue(double *lane_ops_per_s_host, void *stream)
{
    if (!lane_ops_per_s_host) return FOF_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return FOF_ERR_CUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return FOF_ERR_CUDA;
    float *out = nullptr;
    if (cudaMalloc(&out, 256) != cudaSuccess) return FOF_ERR_CUDA;  // a measurement aid may allocate its own 256 bytes
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int iters = 1 << 15, grid = sms * 8;
    double best = 0.0;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0, s);
        fp32_issue_kernel<<<grid, 256, 0, s>>>(out, iters, 1.0000001f, 1e-7f);
        cudaEventRecord(e1, s);
        if (cudaEventSynchronize(e1) != cudaSuccess) break;
        float ms = 0.0f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double ops = (double)grid * 256.0 * (double)iters * kChains * 2.0;
        if (rep > 0 && ms > 0.0f) best = fmax(best, ops / (ms * 1e-3));
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    *lane_ops_per_s_host = best;
    return cudaGetLastError() == cudaSuccess && best > 0.0 ? FOF_OK : FOF_ERR_CUDA;
}

int fof_measure_scatter(const void *in, void *out, int64_t n_records, int32_t log2_window, int32_t scatter_stores,
                        double *records_per_s_host, void *stream)
{
    if (!in || !out || !records_per_s_host || n_records < 4096 || log2_window < 0 || log2_window > 30)
        return FOF_ERR_INVALID_ARG;
    if ((((uintptr_t)in | (uintptr_t)out) & 15) != 0) return FOF_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    const int64_t n = n_records & ~(int64_t)1023;
    if (((int64_t)1 << log2_window) > n) return FOF_ERR_INVALID_ARG;
    const unsigned int wmask = (1u << log2_window) - 1u;
    const unsigned int grid = (unsigned int)(n / 1024);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    double best = 0.0;
    for (int rep = 0; rep < 6; ++rep) {
        cudaEventRecord(e0, s);
        if (scatter_stores) scramble_kernel<true><<<grid, 256, 0, s>>>((const float4 *)in, (float4 *)out, n, wmask);
        else scramble_kernel<false><<<grid, 256, 0, s>>>((const float4 *)in, (float4 *)out, n, wmask);
        cudaEventRecord(e1, s);
        if (cudaEventSynchronize(e1) != cudaSuccess) break;
        float ms = 0.0f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms > 0.0f) best = fmax(best, (double)n / (ms * 1e-3));
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *records_per_s_host = best;
    return cudaGetLastError() == cudaSuccess && best > 0.0 ? FOF_OK : FOF_ERR_CUDA;
}

}  // extern "C"
