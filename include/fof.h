/*
 * fof.h — C ABI of the B200-native periodic Friends-of-Friends library (libfof_b200.so).
 *
 * The calls follow the paper's problem statement: inputs X in R^{N x 3}, box L, linking length b
 * -> labels l in {0..N-1}^N, compact ids, per-group sizes (Alg. 1 input/output;
 * PAPER.md:189-192 Alg. 2 input/output; "Compaction"); everything stays on the
 * device.  PAPER.md = the paper text (arxiv 2510.26851) this repo was built from.
 *
 * Conventions
 *  - "dev" pointers are CUDA device pointers on the current device, "host" pointers are host
 *    memory.  The library never allocates device memory: the caller owns every buffer (PyTorch
 *    tensors in the Python binding) and passes one workspace of fof_workspace_bytes() bytes,
 *    256-byte aligned.  `stream` is a cudaStream_t passed as void* (NULL = default stream).
 *  - Every call returns FOF_OK (0) or a negative FOF_ERR_* code; no exceptions, no abort, no
 *    output on stdout/stderr.
 *  - Particle index type is int32 (N < 2^31).  Positions are float32, row-major [N,3]
 *    (PAPER.md:121, 189), any finite value (they are wrapped into [0,L); a coordinate beyond about
 *    2^24 L in magnitude, where float32 can no longer resolve L, wraps to 0).
 *  - There is NO CPU fallback.  Without a CUDA device the compute calls return FOF_ERR_CUDA.
 */
#ifndef FOF_B200_H
#define FOF_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FOF_OK 0
#define FOF_ERR_INVALID_ARG (-1)  /* NULL pointer, N < 0, N >= 2^31, L <= 0, b <= 0, N_min < 1, ... */
#define FOF_ERR_UNSUPPORTED (-2)  /* fewer than 3 cells of side >= b fit per axis (b > ~L/3)           */
#define FOF_ERR_CUDA (-3)         /* a CUDA runtime call failed (no device, launch error, ...)        */
#define FOF_ERR_NONFINITE (-4)    /* a position was NaN/Inf (deferred: reported by fof_status)        */
#define FOF_ERR_CAPACITY (-5)     /* more kept groups than `cap`; outputs are not valid               */
#define FOF_ERR_STATE (-6)        /* call order violated (e.g. fof_link_stats before fof_link)        */

typedef struct fof_handle fof_handle;

/* Eq. 1: l_link = b_frac * (V/N)^(1/3) with V = L^3, evaluated in double and
 * rounded once to float32.  Host only. */
float fof_linking_length(float b_frac, float L, int64_t N);

/* H0 plan (host only; "Grid setup", with cell side >= b instead of <= b, see
 * DESIGN.md R3).  N particles in a periodic cubic box of side L; `b` is the PHYSICAL linking
 * length in the units of L (Alg. 2 input "linking length b"); groups with fewer
 * than N_min members are dropped by fof_groups ("mass cut", 369).
 * Chooses n cells per axis: n = min(floor(L / (b * 1.001)), ~cbrt(N)) and requires n >= 3.
 * The handle owns host-side plan data only; *out is untouched on error. */
int fof_create(int64_t N, float L, float b, int32_t N_min, fof_handle **out);
void fof_destroy(fof_handle *h);

/* Tuning knob that cannot change results: force n cells per axis (3 <= n <= n_max where
 * n_max = floor(L / (b * 1.001)), n <= 1024).  Changes fof_workspace_bytes(). */
int fof_set_grid(fof_handle *h, int32_t n);
/* n per axis, total cells n^3, largest admissible n. Any out pointer may be NULL. */
int fof_get_grid(const fof_handle *h, int32_t *n, int64_t *cells, int32_t *n_max);

/* Which of the two implementations of H1-H5 fof_link runs (a tuning knob: results are identical).
 *   FOF_PATH_BLOCKS the BLOCK path where the plan admits it (>= 3 blocks of 2^k cells per axis): one
 *                   partition pass into spatial blocks + ghost copies, one CTA per block links out of
 *                   shared memory.  If some block holds more records than a CTA can keep (decided on the
 *                   device, no host synchronisation), the CELL path runs instead, in the same call.
 *   FOF_PATH_CELLS  always the CELL path: two-level counting sort into global cell-contiguous arrays and
 *                   the persistent link kernel over them.  fof_link_stochastic[_batch] and the grid_pairs
 *                   counter of fof_link_stats need those arrays, i.e. a plan set to FOF_PATH_CELLS (or one
 *                   that does not admit the block path).
 *   FOF_PATH_AUTO   (default) the faster of the two for this plan as measured on B200. */
#define FOF_PATH_AUTO 0
#define FOF_PATH_CELLS 1
#define FOF_PATH_BLOCKS 2
int fof_set_path(fof_handle *h, int32_t path);
/* Which path the last fof_link on (h, ws) took (FOF_PATH_BLOCKS or FOF_PATH_CELLS), how many blocks the plan
 * has (0: it does not admit the block path) and the record count of the fullest block (0 if not measured).
 * Any out pointer may be NULL.  Synchronises `stream`. */
int fof_link_path(fof_handle *h, void *ws, void *stream, int32_t *path_host, int32_t *blocks_host,
                  int32_t *max_block_host);

/* Bytes of device workspace fof_link / fof_groups need for this plan (0 on NULL handle). */
size_t fof_workspace_bytes(const fof_handle *h);

/* H1-H5: wrap + bin, cell histogram + exclusive scan (replaces the binary
 * searches of PAPER.md:203-206), cell-contiguous reorder, half-stencil pair
 * tests with the float32 minimum-image predicate d^2 <= b^2 hooked into a
 * lock-free union-find (fixed point of the label sweeps PAPER.md:221-225), flatten.
 *   pos    dev [N,3] float32, read only.
 *   labels dev [N] int32, written: labels[i] = minimum ORIGINAL index of the particles in i's
 *          connected component ("initial label = own index", "minimum
 *          label"), so labels[labels[i]] == labels[i] <= i.
 *   ws     dev workspace, >= fof_workspace_bytes(h), 256-B aligned; contents are scratch.
 * Asynchronous on `stream`; no host synchronisation.  A non-finite position sets a device flag
 * (read it with fof_status); labels are then unspecified but in range. */
int fof_link(fof_handle *h, const float *pos, int32_t *labels, void *ws, void *stream);

/* Counters of the last fof_link on (h, ws): true edges E (unordered pairs with d^2 <= b^2; equal
 * to the oracle's E), distance tests executed (after the geometric reach filter), and the
 * candidate pairs the unfiltered half stencil implies on this plan's grid (P_exec of DESIGN.md §7; 0 unless the
 * plan is set to FOF_PATH_CELLS, see fof_set_path).
 * Any out pointer may be NULL.  Synchronises `stream`. */
int fof_link_stats(fof_handle *h, void *ws, void *stream, uint64_t *edges_host, uint64_t *pair_tests_host,
                   uint64_t *grid_pairs_host);

/* H6-H8: group sizes ("parallel histogram"), compaction of groups with
 * size >= N_min in ascending canonical label, masses and periodic centres
 * of mass (Eq. 4 PAPER.md:259 made periodic: unwrap members relative to the canonical particle,
 * mass-weighted mean in float64, re-wrap into [0,L); R11).
 *   pos, labels     dev, as in fof_link (labels must be canonical: labels[labels[i]] == labels[i]).
 *   mass            dev [N] float32 or NULL (= 1.0 each; "halo mass = particle number").
 *   group_label     dev [cap] int32   canonical label of kept group k (ascending in k)
 *   group_size      dev [cap] int32   member count
 *   group_mass      dev [cap] float32 sum of member masses
 *   group_com       dev [cap,3] float32 periodic centre of mass in [0,L)
 *   particle_group  dev [N] int32 or NULL: compact id of each particle's group, -1 if dropped
 *   cap             capacity of the group_* arrays; floor(N / N_min) always suffices
 *   K_host          host: number of kept groups
 * Synchronises `stream` once to return K.  K > cap -> FOF_ERR_CAPACITY.
 * fof_groups works from (pos, labels) alone.  If `labels` is the very buffer the last fof_link on (h, ws)
 * filled, the group sizes that call counted on the way (H6 is fused into its label pass) are re-used: the
 * caller must then not have modified that buffer in between (pass a copy to have any other labels counted). */
int fof_groups(fof_handle *h, const float *pos, const float *mass, const int32_t *labels, void *ws,
               int32_t *group_label, int32_t *group_size, float *group_mass, float *group_com,
               int32_t *particle_group, int64_t cap, int64_t *K_host, void *stream);

/* Stochastic-edge FoF, one Monte Carlo sample (section 3.2, Eq. 6-8; R25-R28).
 * Every pair of particles closer than the plan's linking length (fof_create's `b`, here the
 * CANDIDATE radius) is a potential edge, kept with probability
 *     p = sigma(alpha (b_link^2 - d^2) / b_link^2),   0 < b_link <= b,
 * (sigma: logistic by a fixed float32 recipe; the decision u < p uses a counter-based generator
 * keyed on (seed, sample, the pair's original indices), so it does not depend on the device or
 * the traversal).  Must follow a fof_link on the same (h, ws): it re-uses that call's cell-sorted
 * arrays, so S samples share one binning; it overwrites the union-find state and the counters of
 * fof_link_stats (edges = sampled edges, pair tests = potential edges of this sample).
 *   labels    dev [N] int32, written: minimum original index of the particle's component in the
 *             sampled graph.
 *   logp      dev, one float64, written: log p(y) = sum over potential edges of
 *             y log p + (1 - y) log(1 - p).
 *   grad_pos  dev [N,3] float32 or NULL: d log p(y) / d pos (the score function of Eq. 7).
 * Asynchronous on `stream`.  FOF_ERR_STATE without a preceding fof_link on (h, ws). */
int fof_link_stochastic(fof_handle *h, float b_link, float alpha, uint64_t seed, uint32_t sample, int32_t *labels,
                        double *logp, float *grad_pos, void *ws, void *stream);

/* S samples sample .. sample + S - 1 of the same step in one call (section 3.2: the S Monte Carlo
 * samples of one REINFORCE step share the neighbour structure).  Candidate filter, distance tests and
 * p_ij are evaluated once for four samples at a time; sample k gives exactly the labels, log p and
 * (to float32 summation order) the score function that fof_link_stochastic(sample + k) gives.
 *   S        1 .. 1024 samples; labels dev [S][N]; logp dev double [S]; grad_pos dev [S][N][3] or NULL.
 *   scratch  dev, fof_stochastic_scratch_bytes(h, S) bytes (one union-find array of N entries per sample), 4-byte
 *            aligned (16-byte alignment and N % 4 == 0 let the label pass use 128-bit loads; neither is required).
 * After the call fof_link_stats reports the potential edges (the same for every sample) as pair tests
 * and the sampled edges summed over the S samples as E.  Same call order rules as fof_link_stochastic.
 * Asynchronous on `stream`. */
size_t fof_stochastic_scratch_bytes(const fof_handle *h, int32_t S);
int fof_link_stochastic_batch(fof_handle *h, float b_link, float alpha, uint64_t seed, uint32_t sample, int32_t S,
                              int32_t *labels, double *logp, float *grad_pos, void *scratch, void *ws, void *stream);

/* The same S samples from a potential-edge LIST ("we do not rebuild the neighbor list"; section 3.2,
 * S = 16 samples per optimisation step share the neighbour structure).  Which pairs are potential
 * edges, their p_ij, t_ij = alpha (b_link^2 - d^2) / b_link^2 and their displacement do not depend on the sample:
 * fof_stochastic_list_build writes them down once per fof_link, and every sample is then one stream over that list
 * (draw, log term, score-function term, hook) instead of a new neighbour search.
 *
 * fof_stochastic_list_build(h, b_link, alpha, list, list_bytes, records_host, ws, stream)
 *   Must follow a fof_link on (h, ws) (FOF_ERR_STATE otherwise; cell path, as fof_link_stochastic).  Counts the
 *   records, synchronises `stream` once to report them in *records_host (every potential edge is recorded under both
 *   of its particles: records = 2 x potential edges), and, if `list` (dev, 256-B aligned, owned by the caller) holds
 *   fof_stochastic_list_bytes(h, *records_host) bytes, fills it (asynchronous on `stream`).  A smaller buffer --
 *   at least fof_stochastic_list_bytes(h, 0), which holds the per-particle offsets -- gives FOF_ERR_CAPACITY with
 *   *records_host set: allocate and call again (the per-particle counts stay in the workspace until the next
 *   fof_link / fof_groups / fof_subgroups on it, so the second call does not search again; they take the place of the
 *   group sizes fof_link left there: a later fof_groups counts its labels afresh).  More than 2^32 - 1 records:
 *   FOF_ERR_CAPACITY as well.
 *   32 bytes per record; at cfg2 (N = 2^24, b = 0.2 spacings as the candidate radius) 2.5e8 records, 8 GB.
 * fof_link_stochastic_list(h, list, seed, sample, S, labels, logp, grad_pos, scratch, ws, stream)
 *   labels / logp / grad_pos / scratch as in fof_link_stochastic_batch, with b_link and alpha those of the build;
 *   sample k gives exactly the labels, and to float32 summation order the log p and score function, of
 *   fof_link_stochastic(sample + k).
 *   `list` must be the buffer of the last fof_stochastic_list_build on h, and no fof_link may have run on h since
 *   (FOF_ERR_STATE): the list describes the positions of the link it was built after.  `ws`: that link's workspace
 *   (only the counters of fof_link_stats are written: pair tests = potential edges, E = sampled edges summed over the
 *   S samples).  Asynchronous on `stream`. */
size_t fof_stochastic_list_bytes(const fof_handle *h, uint64_t records);
int fof_stochastic_list_build(fof_handle *h, float b_link, float alpha, void *list, size_t list_bytes,
                              uint64_t *records_host, void *ws, void *stream);
int fof_link_stochastic_list(fof_handle *h, const void *list, uint64_t seed, uint32_t sample, int32_t S,
                             int32_t *labels, double *logp, float *grad_pos, void *scratch, void *ws, void *stream);

/* Six-dimensional sub-halo pass (section 2.1.1, Eq. 3; R29-R31): inside every
 * kept halo a second FoF in phase space, two members linked iff
 *     (x_i - x_j)^2 / sigma_x + (v_i - v_j)^2 / sigma_v <= ell^2
 * (minimum-image position differences, float32 without FMA).  Downstream of fof_groups:
 * particle_group (dev [N]) and group_size (dev [K]) are its outputs, K its *K_host.
 *   vel         dev [N,3] float32 velocities.
 *   sub_labels  dev [N] int32, written: minimum original index of the particle's 6-D component; a
 *               particle of a dropped halo (particle_group < 0) gets its own index.
 *   ws          the plan's workspace (scratch: the cell-sorted state of fof_link is overwritten, so a
 *               later fof_link_stochastic / fof_link_stats needs a new fof_link first).
 * Work is O(sum over halos of size^2).  Asynchronous on `stream`. */
int fof_subgroups(fof_handle *h, const float *pos, const float *vel, const int32_t *particle_group,
                  const int32_t *group_size, int64_t K, float sigma_x, float sigma_v, float ell, int32_t *sub_labels,
                  void *ws, void *stream);

/* Device steps of the slab-decomposed multi-GPU FoF (section 2.3).  They need
 * no plan; the exchange between devices is done by the caller (paper_2510_26851_b200/slab.py).
 * fof_layer_select: indices i (dev out_idx, capacity N) of the particles whose wrapped coordinate along
 *   `axis` lies in [lo, lo + width) modulo L; *count (dev uint32) = how many; order arbitrary.
 * fof_component_min: out[i] = minimum of ids[] over i's component, given canonical local labels
 *   (labels[labels[i]] == labels[i]); tmp = dev scratch [N].  Turns local labels into the "minimum
 *   global particle ID" of PAPER.md:180.
 * fof_merge_labels: union-find over global ids 0..G-1 (parent = dev scratch [G]), hooked by the P
 *   equivalence pairs (dev [P,2], the smaller id wins), then labels[i] <- root(labels[i]) for the N
 *   labels given (in place).  All asynchronous on `stream`. */
int fof_layer_select(const float *pos, int64_t N, float L, int32_t axis, float lo, float width, int32_t *out_idx,
                     uint32_t *count, void *stream);
int fof_component_min(const int32_t *labels, const int32_t *ids, int64_t N, int32_t *tmp, int32_t *out, void *stream);
int fof_merge_labels(const int32_t *pairs, int64_t P, int32_t *parent, int64_t G, int32_t *labels, int64_t N,
                     void *stream);
/* fof_merge_labels_sparse: the same merge with a union-find over the U DISTINCT labels that occur in the pairs
 *   (uniq: dev [U], ascending; parent: dev scratch [U]) instead of one entry per global id (the
 *   cost of the union step is what made the paper's slab run slow).  Labels that no pair mentions are untouched.
 * fof_combine_groups: cross-rank group construction.  Every rank has run fof_groups on its own particles plus
 *   one massless proxy per canonical particle that lives on another rank, and the partial records of the groups
 *   that touch a ghost layer have been gathered: part_label [P] ASCENDING (dev), part_size [P] members (proxies
 *   not counted), part_mass [P], part_com [P,3].  For each of the W groups `want` [W] whose canonical particle
 *   this rank owns (ref [W,3] = its position) the records with that label are combined into out_size [W],
 *   out_mass [W], out_com [W,3]: mass-weighted mean of the minimum-image displacements from the canonical
 *   particle, re-wrapped (R11), float64.  All asynchronous on `stream`. */
int fof_merge_labels_sparse(const int32_t *pairs, int64_t P, const int32_t *uniq, int64_t U, int32_t *parent,
                            int32_t *labels, int64_t N, void *stream);
int fof_combine_groups(const int32_t *want, int64_t W, const float *ref, float L, const int32_t *part_label, int64_t P,
                       const int32_t *part_size, const float *part_mass, const float *part_com, int32_t *out_size,
                       float *out_mass, float *out_com, void *stream);

/* Halo decoration (section 3.1.1 "Decorated Frozen Assignment": "particle standard deviation
 * (sigma)" as the surrogate of halo mass; R23):
 *   group_sigma[k] = sqrt( sum_i m_i |delta_i|^2 / M_k ),  delta_i = minimum-image displacement of
 * member i from group_com[k], accumulated in float64.  Downstream of fof_groups: particle_group,
 * group_mass, group_com are its outputs (dev), K its *K_host.  `ws` as in fof_groups (scratch).
 *   group_sigma  dev [K] float32, written.
 * Asynchronous on `stream`. */
int fof_group_sigma(fof_handle *h, const float *pos, const float *mass, const int32_t *particle_group,
                    const float *group_mass, const float *group_com, int64_t K, void *ws, float *group_sigma,
                    void *stream);

/* fof_group_sigma without a workspace, for callers that cannot allocate one (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc).  Same operation (section 3.1.1, Eq. 5), same kernels,
 * same arguments minus `ws`: the scratch (one float64 accumulator per group) is a file-scope device array of the
 * library, FOF_SIGMA_STATIC_MAX_GROUPS entries = 2 MiB, which every GPU that loads the library holds until the
 * process exits.  The call allocates nothing and frees nothing (no cudaMalloc, cudaFree or allocating library
 * routine; the first call on a device asks the runtime once for the array's device address).
 *   K > FOF_SIGMA_STATIC_MAX_GROUPS -> FOF_ERR_CAPACITY, nothing is launched (use fof_group_sigma);
 *   K > floor(N / N_min) or a missing pointer -> FOF_ERR_INVALID_ARG, as fof_group_sigma.
 * Every call on a device shares that one array: it is cleared on `stream` at the start of each call, so calls one
 * after the other on one stream (or otherwise ordered) are independent, but two calls that OVERLAP on the GPU --
 * different streams, different handles, different host threads -- race on it and give wrong sigmas.  Serialise
 * them, or use fof_group_sigma with a workspace per stream.  Asynchronous on `stream`. */
#define FOF_SIGMA_STATIC_MAX_GROUPS 262144
int fof_group_sigma_static(fof_handle *h, const float *pos, const float *mass, const int32_t *particle_group,
                           const float *group_mass, const float *group_com, int64_t K, float *group_sigma,
                           void *stream);

/* Frozen-assignment backward (section 3.1, Eq. 4: dX^h/dtheta = (1/N) sum_i dx_i/dtheta;
 * Eq. 5 for the decoration; R24).  Membership is held fixed:
 *   grad_pos[i] = (m_i / M_k) (grad_com[k] + grad_sigma[k] delta_i / group_sigma[k]),  k = particle_group[i],
 * and 0 for a particle of a dropped group (k < 0); the sigma term is 0 where group_sigma[k] = 0.
 *   grad_com    dev [K,3] float32 dL/dX_k, or NULL (= 0)
 *   grad_sigma  dev [K] float32 dL/dsigma_k, or NULL (= 0; then group_sigma may be NULL too)
 *   grad_pos    dev [N,3] float32, written (every element).
 * Asynchronous on `stream`; needs no workspace. */
int fof_groups_backward(fof_handle *h, const float *pos, const float *mass, const int32_t *particle_group,
                        const float *group_mass, const float *group_com, const float *group_sigma,
                        const float *grad_com, const float *grad_sigma, int64_t K, float *grad_pos, void *stream);

/* Host-buffer entry point (the end-to-end call): copies pos (and mass) host -> device, runs
 * fof_link + fof_groups, copies labels and the K group records device -> host.
 *   *_host  host buffers (pinned for full copy speed); mass_host / particle_group_host may be NULL.
 *   dev_buf device scratch of fof_host_device_bytes(h, cap) bytes, 256-B aligned.
 * The labels are copied back on an internal stream while the groups are built on `stream`.
 * Synchronises `stream` (and that copy) before it returns. */
size_t fof_host_device_bytes(const fof_handle *h, int64_t cap);
int fof_run_host(fof_handle *h, const float *pos_host, const float *mass_host, int32_t *labels_host,
                 int32_t *group_label_host, int32_t *group_size_host, float *group_mass_host,
                 float *group_com_host, int32_t *particle_group_host, int64_t cap, int64_t *K_host,
                 void *dev_buf, void *stream);

/* The same work as fof_run_host, split into an enqueue half and a completion half so that a SEQUENCE of inputs
 * (the "simulation analysis" use of PAPER.md:14 with the snapshots on the host: one catalogue per snapshot) keeps the PCIe link busy in
 * both directions: while input k is linked, input k+1 travels host -> device and result k-1 device -> host.
 * Three internal streams (in, run, out) order the work; the caller's streams are not involved.
 *   slot      0 or 1.  At most one submit is outstanding per slot (else FOF_ERR_STATE); each slot has its own
 *             dev_buf of fof_host_device_bytes(h, cap) bytes (256-B aligned), owned by the caller, which must not
 *             touch it between the submit and the wait.
 *   *_host    as in fof_run_host; pinned memory is REQUIRED for the overlap (pageable copies serialise).  They
 *             must stay valid, and the outputs unread, until fof_host_wait(h, slot) returns.
 * fof_host_submit returns once the copies and kernels are enqueued (it does not block on the device; inputs of
 * consecutive submits are processed in submit order).  fof_host_wait blocks until the slot's labels, K group
 * records and particle_group are in the host buffers, writes *K_host, frees the slot and returns the deferred
 * status: FOF_OK, FOF_ERR_NONFINITE, FOF_ERR_CAPACITY (K > cap: *K_host is set, no group record is copied), or
 * FOF_ERR_STATE if the slot has no submit outstanding or its submit had failed.  fof_destroy waits for whatever
 * is still in flight.  Results are those of fof_run_host bit for bit. */
int fof_host_submit(fof_handle *h, int32_t slot, const float *pos_host, const float *mass_host, int32_t *labels_host,
                    int32_t *group_label_host, int32_t *group_size_host, float *group_mass_host,
                    float *group_com_host, int32_t *particle_group_host, int64_t cap, void *dev_buf);
int fof_host_wait(fof_handle *h, int32_t slot, int64_t *K_host);

/* Synchronises `stream` and returns the deferred device-side status of the last fof_link /
 * fof_groups on (h, ws): FOF_OK or FOF_ERR_NONFINITE. */
int fof_status(fof_handle *h, void *ws, void *stream);

/* Measurement aids (they never change results).
 * fof_profile_enable(h, slots): slots > 0 makes fof_link / fof_groups record a CUDA event on
 * `stream` before and after every stage (one kernel launch or one memset group each), into one of
 * `slots` event sets used round-robin, one set per fof_link call (and the fof_groups calls that
 * follow it); slots = 0 switches profiling off.  fof_profile_read synchronises the recorded events
 * and returns, for each stage k < fof_profile_count(h), the MEAN device time in milliseconds over
 * the sets recorded since the previous read (0 for a stage that did not run), then forgets them.
 * fof_profile_name(h, k) is a static string ("link.bin", "groups.reduce", ...).
 * fof_launch_count: kernels this handle has launched so far (memsets and copies not counted). */
int fof_profile_enable(fof_handle *h, int slots);
/* Restrict the recorded events to stage `stage` (0 <= stage < fof_profile_count), or -1 for every stage
 * (the default): two events per step instead of two per stage keep the timed region undisturbed. */
int fof_profile_only(fof_handle *h, int stage);
int fof_profile_count(const fof_handle *h);
const char *fof_profile_name(const fof_handle *h, int k);
int fof_profile_read(fof_handle *h, float *ms, int cap);
uint64_t fof_launch_count(const fof_handle *h);

/* Measured ceilings (measurement aids; they run no step of the method).
 * fof_measure_fp32_issue: FP32 lane-operations per second of this device on a non-FMA FADD + FMUL stream (the
 *   instruction mix of the link predicate, which forbids FMA contraction), best of four timed launches that
 *   fill every SM; the ceiling bench.py quotes for the ALU-bound link kernel.  Allocates
 *   (and frees) 256 bytes of device memory of its own.
 * fof_measure_scatter: records per second of a copy of n_records 16-byte records (dev in/out, 16-byte aligned,
 *   n_records >= 4096) in which the stores (scatter_stores != 0) or the loads are scattered inside windows of
 *   2^log2_window records and the other side is coalesced: the floor of a reorder pass of H3.
 * Both synchronise `stream`. */
int fof_measure_fp32_issue(double *lane_ops_per_s_host, void *stream);
int fof_measure_scatter(const void *in, void *out, int64_t n_records, int32_t log2_window, int32_t scatter_stores,
                        double *records_per_s_host, void *stream);

/* Static string for an error code. */
const char *fof_error_string(int code);

/* Text of the last CUDA runtime error seen by this handle ("" if none). */
const char *fof_last_cuda_error(const fof_handle *h);

#ifdef __cplusplus
}
#endif
#endif /* FOF_B200_H */
