// kernels_noalloc.cu — fof_group_sigma_static: the halo decoration of fof_group_sigma (PAPER.md:283-290 section
// 3.1.1, Eq. 5) for callers that cannot hand the library a workspace they allocated: code under
// CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The same two kernels as fof_group_sigma
// (sigma_accum_kernel, sigma_finish_kernel, through launch_group_sigma); the only difference is where their scratch --
// one float64 accumulator per group -- lives: in the file-scope device array below instead of the caller's workspace.
//
// The array's name is a host-side stand-in in host code, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress, asked once per device with that device current.  Every GPU that loads the library holds the
// array (FOF_SIGMA_STATIC_MAX_GROUPS x 8 bytes = 2 MiB) until the process exits.
#include <cstdio>
#include <mutex>

#include "fof_internal.cuh"

namespace {

constexpr int64_t kStaticGroups = FOF_SIGMA_STATIC_MAX_GROUPS;

static __device__ __align__(256) double g_sigma_acc[kStaticGroups];

constexpr int kMaxDevices = 64;
double *g_acc_addr[kMaxDevices];  // device address of g_sigma_acc on device d; null until asked for
std::mutex g_acc_mutex;

// The device address of g_sigma_acc on the CURRENT device (set-up on the first call per device; no allocation:
// the array is part of the module image).
cudaError_t static_acc_address(double **out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_acc_mutex);
    if (!g_acc_addr[dev]) {
        double *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_sigma_acc);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_acc_addr[dev] = p;
    }
    *out = g_acc_addr[dev];
    return cudaSuccess;
}

int fail(fof_handle *h, cudaError_t e, const char *where)
{
    snprintf(h->cuda_err, sizeof(h->cuda_err), "%s: %s", where, cudaGetErrorString(e));
    (void)cudaGetLastError();
    return FOF_ERR_CUDA;
}

}  // namespace

extern "C" int fof_group_sigma_static(fof_handle *h, const float *pos, const float *mass, const int32_t *particle_group,
                                      const float *group_mass, const float *group_com, int64_t K, float *group_sigma,
                                      void *stream)
{
    if (!h || K < 0 || K > h->max_groups) return FOF_ERR_INVALID_ARG;
    if (K > kStaticGroups) return FOF_ERR_CAPACITY;  // more groups than the static scratch holds: use fof_group_sigma
    if (h->N > 0 && (!pos || !particle_group)) return FOF_ERR_INVALID_ARG;
    if (K > 0 && (!group_mass || !group_com || !group_sigma)) return FOF_ERR_INVALID_ARG;
    if (K == 0) return FOF_OK;
    double *acc = nullptr;
    cudaError_t e = static_acc_address(&acc);
    if (e != cudaSuccess) return fail(h, e, "fof_group_sigma_static: cudaGetSymbolAddress");
    h->launches += 2;
    // launch_group_sigma clears acc[0 .. K) on `stream` first: the array keeps the previous call's sums
    e = fof::launch_group_sigma(pos, mass, particle_group, h->N, h->grid, group_mass, group_com, K, acc, group_sigma,
                                (cudaStream_t)stream);
    if (e != cudaSuccess) return fail(h, e, "sigma kernels (static scratch)");
    return FOF_OK;
}
