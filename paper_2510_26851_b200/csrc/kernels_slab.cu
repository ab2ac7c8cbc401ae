// kernels_slab.cu — device steps of the slab-decomposed multi-GPU FoF.
// PAPER.md:176-182 (section 2.3): the box is cut into slabs along one axis; every device links its slab
// plus a ghost layer at least b thick borrowed from its neighbour, the labels of the ghost particles
// give label equivalences between neighbouring devices, one union-find over those equivalences
// merges them, and every particle is relabelled to the "minimum global particle ID" of its group
// (PAPER.md:180).  The exchange itself (ring send/recv of the ghost layer, all-gather of the
// equivalence pairs) is torch.distributed plumbing in paper_2510_26851_b200/slab.py; the steps here
// are the ones that touch every particle or every pair:
//   layer_select_kernel    indices of the particles inside a layer [z_lo, z_lo + width) (periodic)
//   component_min_kernels  canonical label in GLOBAL ids: min over the local component of ids[]
//   merge kernels          dense union-find over global ids (parent[g] = g initially), hooked by the
//                          equivalence pairs with atomicMin-free CAS on roots (smaller id wins), then
//                          labels[i] <- root(labels[i])
#include "fof_internal.cuh"

namespace fof {

__global__ void __launch_bounds__(kBlock) layer_select_kernel(const float *__restrict__ pos, int64_t N, float L,
                                                              int axis, float lo, float width,
                                                              int *__restrict__ out_idx, unsigned int *count)
{
    const int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    bool in = false;
    if (i < N) {
        const float w = wrap1(__ldg(pos + 3 * i + axis), L);
        float d = __fsub_rn(w, lo);
        if (d < 0.0f) d = __fadd_rn(d, L);
        in = d < width;
    }
    // warp-aggregated append (order inside the list is arbitrary)
    const unsigned int bal = __ballot_sync(0xffffffffu, in);
    if (bal == 0u) return;
    const int lane = threadIdx.x & 31;
    unsigned int base = 0;
    if (lane == __ffs((int)bal) - 1) base = atomicAdd(count, (unsigned int)__popc(bal));
    base = __shfl_sync(0xffffffffu, base, __ffs((int)bal) - 1);
    if (in) out_idx[base + __popc(bal & ((1u << lane) - 1u))] = (int)i;
}

// tmp[labels[i]] = min over the component of ids; out[i] = tmp[labels[i]].  labels are canonical
// local labels (labels[labels[i]] == labels[i]), so tmp is only touched at canonical particles.
__global__ void __launch_bounds__(kBlock) component_min_init_kernel(const int *__restrict__ labels,
                                                                    const int *__restrict__ ids, int64_t N,
                                                                    int *__restrict__ tmp)
{
    const int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (i < N && labels[i] == (int)i) tmp[i] = ids[i];
}

__global__ void __launch_bounds__(kBlock) component_min_reduce_kernel(const int *__restrict__ labels,
                                                                      const int *__restrict__ ids, int64_t N,
                                                                      int *tmp)
{
    const int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (i < N && labels[i] != (int)i) atomicMin(tmp + labels[i], ids[i]);
}

__global__ void __launch_bounds__(kBlock) component_min_gather_kernel(const int *__restrict__ labels, int64_t N,
                                                                      const int *__restrict__ tmp,
                                                                      int *__restrict__ out)
{
    const int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (i < N) out[i] = tmp[labels[i]];
}

// ---- dense union-find over global ids: parent[g] <= g, roots have parent[g] == g --------------
__global__ void __launch_bounds__(kBlock) iota_parent_kernel(int *__restrict__ parent, int64_t G)
{
    const int64_t g = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (g < G) parent[g] = (int)g;
}

__device__ __forceinline__ int find_dense(int *parent, int x)
{
    int p = parent[x];
    while (p != x) {
        const int gp = parent[p];
        if (gp != p) parent[x] = gp;  // halve
        x = p;
        p = gp;
    }
    return x;
}

__global__ void __launch_bounds__(kBlock) merge_pairs_kernel(const int *__restrict__ pairs, int64_t P, int *parent)
{
    const int64_t k = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (k >= P) return;
    int ra = find_dense(parent, pairs[2 * k]), rb = find_dense(parent, pairs[2 * k + 1]);
    while (ra != rb) {
        if (ra < rb) { const int t = ra; ra = rb; rb = t; }  // ra is the larger root: it hooks under rb
        const int old = atomicCAS(parent + ra, ra, rb);
        if (old == ra) break;
        ra = find_dense(parent, old);
    }
}

__global__ void __launch_bounds__(kBlock) relabel_kernel(int *__restrict__ labels, int64_t N, int *parent)
{
    const int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (i >= N) return;
    int x = labels[i];
    while (parent[x] != x) x = parent[x];
    labels[i] = x;
}

// ---- sparse variant: the union-find runs over the U DISTINCT labels that occur in the equivalence pairs
// (uniq, ascending), not over all global ids; a label is found by binary search. ------------------------
__device__ __forceinline__ int lower_bound_i32(const int *__restrict__ a, int n, int key)
{
    int lo = 0, hi = n;
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (__ldg(a + mid) < key) lo = mid + 1;
        else hi = mid;
    }
    return lo;
}

// hooks by VALUE of the label (the smaller global id wins), parent holds positions in uniq
__global__ void __launch_bounds__(kBlock) merge_pairs_sparse_kernel(const int *__restrict__ pairs, int64_t P,
                                                                    const int *__restrict__ uniq, int U, int *parent)
{
    const int64_t k = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (k >= P) return;
    // uniq is ascending, so "smaller position" == "smaller label": the dense hook rule applies to positions
    int ra = find_dense(parent, lower_bound_i32(uniq, U, pairs[2 * k]));
    int rb = find_dense(parent, lower_bound_i32(uniq, U, pairs[2 * k + 1]));
    while (ra != rb) {
        if (ra < rb) { const int t = ra; ra = rb; rb = t; }
        const int old = atomicCAS(parent + ra, ra, rb);
        if (old == ra) break;
        ra = find_dense(parent, old);
    }
}

__global__ void __launch_bounds__(kBlock) relabel_sparse_kernel(int *__restrict__ labels, int64_t N,
                                                                const int *__restrict__ uniq, int U, int *parent)
{
    const int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (i >= N) return;
    const int l = labels[i];
    int x = lower_bound_i32(uniq, U, l);
    if (x >= U || __ldg(uniq + x) != l) return;  // a label no pair mentions: nothing to merge
    while (parent[x] != x) x = parent[x];
    labels[i] = __ldg(uniq + x);
}

// ---- cross-rank group construction (H6-H8 over slabs): every rank has run fof_groups on its own particles
// plus one massless PROXY per canonical particle that lives on another rank (so that its members are unwrapped
// relative to the same reference as in a monolithic run), and the partial records (label, members, mass, centre
// of mass) of the groups that touch a ghost layer have been gathered, sorted by label.  The owner of the
// canonical particle of such a group combines them:
//   size = sum of members,  M = sum of partial masses,
//   com = wrap(r + sum_k M_k minimg(c_k - r) / M),  r = wrapped position of the canonical particle:
// minimg(c_k - r) is the mean displacement of rank k's members (|mean| <= L/2), so this is the mass-weighted
// mean of ALL members' minimum-image displacements from r, the definition of DESIGN.md R11. -------------------
__global__ void __launch_bounds__(kBlock) combine_groups_kernel(const int *__restrict__ want, int64_t W,
                                                                const float *__restrict__ ref, float L,
                                                                const int *__restrict__ part_label, int64_t P,
                                                                const int *__restrict__ part_size,
                                                                const float *__restrict__ part_mass,
                                                                const float *__restrict__ part_com,
                                                                int *__restrict__ out_size, float *__restrict__ out_mass,
                                                                float *__restrict__ out_com)
{
    const int64_t k = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (k >= W) return;
    const int lab = want[k];
    const double Ld = (double)L, h = 0.5 * (double)L;
    const double r[3] = {(double)wrap1(ref[3 * k], L), (double)wrap1(ref[3 * k + 1], L), (double)wrap1(ref[3 * k + 2], L)};
    double M = 0.0, s[3] = {0.0, 0.0, 0.0};
    long long n = 0;
    for (int64_t j = lower_bound_i32(part_label, (int)P, lab); j < P && part_label[j] == lab; ++j) {
        const double m = (double)part_mass[j];
        n += part_size[j];
        M += m;
        for (int a = 0; a < 3; ++a) {
            double d = (double)part_com[3 * j + a] - r[a];
            if (d > h) d -= Ld;
            else if (d < -h) d += Ld;
            s[a] += m * d;
        }
    }
    out_size[k] = (int)n;
    out_mass[k] = (float)M;
    for (int a = 0; a < 3; ++a) {
        double c = r[a] + (M > 0.0 ? s[a] / M : 0.0);
        if (c < 0.0) c += Ld;
        if (c >= Ld) c -= Ld;
        float cf = (float)c;
        if (cf >= L) cf = 0.0f;
        out_com[3 * k + a] = cf;
    }
}

static inline unsigned int blocks_for(int64_t n) { return (unsigned int)((n + kBlock - 1) / kBlock); }

cudaError_t launch_merge_labels_sparse(const int *pairs, int64_t P, const int *uniq, int64_t U, int *parent, int *labels,
                                       int64_t N, cudaStream_t s)
{
    if (U > 0) iota_parent_kernel<<<blocks_for(U), kBlock, 0, s>>>(parent, U);
    if (P > 0 && U > 0) merge_pairs_sparse_kernel<<<blocks_for(P), kBlock, 0, s>>>(pairs, P, uniq, (int)U, parent);
    if (N > 0 && U > 0) relabel_sparse_kernel<<<blocks_for(N), kBlock, 0, s>>>(labels, N, uniq, (int)U, parent);
    return cudaGetLastError();
}

cudaError_t launch_combine_groups(const int *want, int64_t W, const float *ref, float L, const int *part_label, int64_t P,
                                  const int *part_size, const float *part_mass, const float *part_com, int *out_size,
                                  float *out_mass, float *out_com, cudaStream_t s)
{
    if (W > 0)
        combine_groups_kernel<<<blocks_for(W), kBlock, 0, s>>>(want, W, ref, L, part_label, P, part_size, part_mass,
                                                               part_com, out_size, out_mass, out_com);
    return cudaGetLastError();
}

cudaError_t launch_layer_select(const float *pos, int64_t N, float L, int axis, float lo, float width, int *out_idx,
                                unsigned int *count, cudaStream_t s)
{
    cudaError_t e = cudaMemsetAsync(count, 0, sizeof(unsigned int), s);
    if (e != cudaSuccess) return e;
    if (N > 0) layer_select_kernel<<<blocks_for(N), kBlock, 0, s>>>(pos, N, L, axis, lo, width, out_idx, count);
    return cudaGetLastError();
}

cudaError_t launch_component_min(const int *labels, const int *ids, int64_t N, int *tmp, int *out, cudaStream_t s)
{
    if (N <= 0) return cudaSuccess;
    component_min_init_kernel<<<blocks_for(N), kBlock, 0, s>>>(labels, ids, N, tmp);
    component_min_reduce_kernel<<<blocks_for(N), kBlock, 0, s>>>(labels, ids, N, tmp);
    component_min_gather_kernel<<<blocks_for(N), kBlock, 0, s>>>(labels, N, tmp, out);
    return cudaGetLastError();
}

cudaError_t launch_merge_labels(const int *pairs, int64_t P, int *parent, int64_t G, int *labels, int64_t N,
                                cudaStream_t s)
{
    if (G > 0) iota_parent_kernel<<<blocks_for(G), kBlock, 0, s>>>(parent, G);
    if (P > 0) merge_pairs_kernel<<<blocks_for(P), kBlock, 0, s>>>(pairs, P, parent);
    if (N > 0) relabel_kernel<<<blocks_for(N), kBlock, 0, s>>>(labels, N, parent);
    return cudaGetLastError();
}

}  // namespace fof
