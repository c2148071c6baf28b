/* sdm.h -- C ABI of libsdm: one Super-Droplet Method (SDM) coalescence timestep on one B200.
 *
 * Method: Bartman & Arabas, "On the design of Monte-Carlo particle coagulation solver interface:
 * a CPU/GPU Super-Droplet Method case study with PySDM", arXiv 2101.06318, cited below as
 * PAPER.md:<line>.  State of Fig. 2: per super-droplet a multiplicity xi
 * (int64), one extensive attribute, the volume v (fp64, m^3), and a cell id (int32).  Call order
 * and in/out intents follow Fig. 3.  Readings of the paper where it is silent
 * (RNG stream, tie rules, evaluation order, ...) are R1..R20 of DESIGN.md.
 *
 * Conventions
 *  - Every entry point returns an int status: SDM_OK (0) or a negative SDM_E* code.  Nothing
 *    throws or aborts across this boundary.  sdm_last_error() gives a message for the last failure.
 *  - "_dev" pointers are DEVICE pointers (CUDA global memory of the current device); "_host"
 *    pointers are HOST pointers (pinned memory recommended).  The library NEVER allocates device
 *    memory: the caller supplies one workspace (sdm_workspace_bytes) that must outlive the handle
 *    ("explicit allocation is used only once per simulation").
 *  - All device work is enqueued on the cudaStream_t given to sdm_create.  Calls are asynchronous
 *    with respect to the host unless they return a host value (documented per call).
 *  - User arrays are caller-owned and only read/written during the call (stream order).
 *  - Storage order is observable (it feeds the RNG counter and the exported permutation): it is
 *    the order given to sdm_set_state, then changed only by the stable compaction sdm_remove_zero.
 *  - There is no CPU fallback: without a CUDA device every compute call fails with SDM_ECUDA.
 */
#ifndef SDM_H
#define SDM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sdm sdm_t; /* opaque handle, owned by the library (host memory only) */

enum { SDM_OK = 0, SDM_EINVAL = -1, SDM_ECAPACITY = -2, SDM_ECUDA = -3, SDM_ESTATE = -4 };

/* Coalescence kernel a(v1, v2) of Eq. 1 / Eq. 3. */
enum { SDM_KERNEL_GOLOVIN = 0, SDM_KERNEL_GRAVITATIONAL = 1, SDM_KERNEL_GRAVITATIONAL_TABULATED = 2,
       SDM_KERNEL_USER = 3 /* a(v1, v2) from caller-supplied CUDA source, sdm_set_kernel_source; b and E are ignored */ };
typedef struct {
    int32_t type;     /* SDM_KERNEL_*                                                              */
    int32_t reserved; /* must be 0                                                                 */
    double b;         /* Golovin: a = b*(v1+v2), b in 1/s                           */
    double E;         /* gravitational: a = E*pi*(r1+r2)^2*|w(r1)-w(r2)|, collection efficiency E  */
                      /* (constants of BASELINE.json config 3, R9-R10)      */
                      /* tabulated: a = E*Etab(r1,r2)*pi*(r1+r2)^2*|w(r1)-w(r2)|, Etab from              */
                      /* sdm_set_efficiency_table                                                     */
} sdm_kernel_t;

/* Options for sdm_set_option (testing / profiling; defaults in brackets). */
enum {
    SDM_OPT_FORCE_GENERAL = 1, /* [0] 1: never take the cell-contiguous fused path                 */
    SDM_OPT_SEGMENT_CAP = 2,   /* [0] >0: override the largest segment a warp sorts on chip (tests) */
    SDM_OPT_WRITE_IDX = 3,     /* [1] 0: do not export the permutation (idx is then undefined)      */
    SDM_OPT_SCREENING = 4,     /* [1] 0: evaluate Eq. 3 in fp64 for every pair (no fp32 pre-test)   */
    SDM_OPT_TIMING = 5,        /* [0] 1: bracket the dominant kernel of each step with CUDA events   */
    SDM_OPT_LANES_PER_CELL = 6, /* [0] 16: 16 lanes x 16 droplets for cells of 129..256 (tuning)         */
    SDM_OPT_SORT_ENGINE = 7,   /* [0] fused path, per-cell permutation: 0 automatic (counting sort on the */
                               /*     top key bits when no cell exceeds 256 droplets -- small cells in    */
                               /*     groups of up to 8 -- else the register sorting network), 1 the      */
                               /*     network, 2 the counting sort (cells <= 256 only)                    */
    SDM_OPT_DETERMINISTIC = 8, /* [0] 1: cells are mapped to warps by a fixed rule (no work tickets), so the  */
                               /*     fp64 moment sums M1, M2 of sdm_coalescence_step_moments are reproducible */
                               /*     bit for bit from run to run (xi, v, idx, M0 always are)                 */
    SDM_OPT_BOX_CTAS = 10,     /* [0] >0: number of CTAs of the persistent box kernel (n_cell == 1; tuning), at   */
                               /*     most the SM count; 0: chosen from the droplet count                          */
    SDM_OPT_BOX_REGION_CAP = 11, /* [0] >0: capacity of a region of the box kernel's record queue (tests: a small value   */
                               /*     forces the overflow fallback to exact region offsets)                             */
    SDM_OPT_BOX_SORT_CAP = 12, /* [0] >0: largest region the box kernel sorts in shared memory (tests: a small value    */
                               /*     forces the ranking-by-counting fallback in global memory)                        */
    SDM_OPT_COOPERATIVE = 13,  /* [1] 0: behave as on a device (or context) without cooperative launches: the compaction */
                               /*     is a plain launch and the next step rebuilds its cell table, single-cell boxes take   */
                               /*     the general path (tests; the library falls back to the same by itself when a         */
                               /*     cooperative grid does not fit, e.g. under MPS)                                        */
    SDM_OPT_CTAS_PER_SM = 9    /* [0] >0: grid of the counting-sort kernel = value x SM count, at most 32      */
                               /*     (scaling runs; SDM_EINVAL if the grid would exceed the moment partials)  */
};

/* Counter slots returned by sdm_get_counters. */
enum {
    SDM_CNT_N_SD = 0,        /* current number of super-droplets                                   */
    SDM_CNT_EVENTS = 1,      /* pairs with gamma_tilde > 0 since sdm_set_state                      */
    SDM_CNT_ZEROS = 2,       /* droplets with xi == 0 currently in the state                        */
    SDM_CNT_LAUNCHES = 3,    /* kernels launched by this handle since sdm_create                    */
    SDM_CNT_MODE = 4,        /* 0 = general path, 1 = fused cell-contiguous path, 2 = single-cell box  */
                             /* path (n_cell == 1: all steps of a call in one persistent launch)      */
    SDM_CNT_MAX_CELL = 5,    /* largest per-cell count seen at sdm_set_state                        */
    SDM_CNT_EXACT_EVALS = 6, /* pairs whose Eq. 3 was evaluated in fp64 since sdm_set_state         */
    SDM_CNT_COUNT = 8
};

/* Bytes of device workspace needed for `capacity` super-droplets in `n_cell` cells; 0 if the
 * arguments are invalid (capacity < 1, capacity > SDM_MAX_CAPACITY, n_cell < 1).  Storage indices are 32-bit
 * inside the kernels; the bound leaves room for the grid-stride loops' last increment. */
#define SDM_MAX_CAPACITY 2139095040 /* 2^31 - 2^23 */
size_t sdm_workspace_bytes(int64_t capacity, int32_t n_cell);

/* The same for a state with n_attr extensive attributes per super-droplet (1 <= n_attr <= SDM_MAX_ATTR):
 * the paper's `attributes = Storage((N_ATTR, N_SD), float)`, a 2-D row-major block whose row 0 is the
 * volume (`volume_view`).  n_attr == 1 equals sdm_workspace_bytes. */
#define SDM_MAX_ATTR 8
size_t sdm_workspace_bytes_attr(int64_t capacity, int32_t n_cell, int32_t n_attr);

/* Creates a handle.  workspace_dev: caller-owned device memory, 256-byte aligned, at least
 * sdm_workspace_bytes(capacity, n_cell) bytes.  cuda_stream: a cudaStream_t (NULL = legacy default
 * stream).  The state is empty (n_sd = 0) until sdm_set_state.  Synchronous (clears the control
 * block).  Errors: SDM_EINVAL (bad arguments, workspace too small or misaligned), SDM_ECUDA. */
int sdm_create(sdm_t **out, int64_t capacity, int32_t n_cell, void *workspace_dev,
               size_t workspace_bytes, void *cuda_stream);

/* sdm_create for n_attr extensive attributes (sdm_create is n_attr = 1); the workspace must hold
 * sdm_workspace_bytes_attr(capacity, n_cell, n_attr) bytes. */
int sdm_create_attr(sdm_t **out, int64_t capacity, int32_t n_cell, int32_t n_attr, void *workspace_dev,
                    size_t workspace_bytes, void *cuda_stream);

/* Frees the handle (host memory only; the workspace stays with the caller).  Synchronises the stream. */
int sdm_destroy(sdm_t *h);

int sdm_set_option(sdm_t *h, int32_t option, int64_t value);

/* Copies a state of n_sd super-droplets into the workspace (Fig. 2: multiplicities, attributes[0],
 * cell_id), validates it (0 <= cell_id < n_cell, xi >= 0, v finite and > 0) and
 * analyses its layout (cell-contiguous or not, largest cell).  SYNCHRONOUS.  Errors: SDM_ECAPACITY
 * (n_sd > capacity), SDM_EINVAL (validation failed; the state is then unusable: SDM_ESTATE later). */
int sdm_set_state(sdm_t *h, int64_t n_sd, const int64_t *xi_dev, const double *v_dev,
                  const int32_t *cell_id_dev);
int sdm_set_state_host(sdm_t *h, int64_t n_sd, const int64_t *xi_host, const double *v_host,
                       const int32_t *cell_id_host);

/* Rows 1 .. n_attr-1 of the attribute block (row 0, the volume, goes through sdm_set_state): row r is read
 * from attr_dev + (r-1)*ld, n_sd values each, ld >= n_sd in elements.  Call it after sdm_set_state, which
 * zero-fills these rows; n_sd is that call's n_sd.  Every value must be finite (else SDM_EINVAL and the
 * state becomes unusable).  The rows are updated by every coalescence event exactly like the volume
 * (Fig. 5 loop over attributes: A_k += g A_j, or both g A_j + A_k on the split branch),
 * move with their droplet in sdm_remove_zero, and never enter Eq. 3.  SYNCHRONOUS.  SDM_EINVAL if the
 * handle has n_attr == 1. */
int sdm_set_attributes(sdm_t *h, const double *attr_dev, int64_t ld);

/* Copies rows 1 .. n_attr-1 out (row r to attr_dev + (r-1)*ld, current n_sd values each).  SYNCHRONOUS. */
int sdm_get_attributes(sdm_t *h, double *attr_dev, int64_t ld);

/* User-supplied collection efficiencies for SDM_KERNEL_GRAVITATIONAL_TABULATED (the paper separates the
 * pair logic from "potentially user-supplied kernel code", and takes its kernels with their
 * efficiencies from tables after Berry 1967): E_host[n_r * n_r], row-major, E_host[i*n_r + k] =
 * efficiency for radii (r_grid_host[i], r_grid_host[k]), on a strictly increasing grid of positive radii [m],
 * 2 <= n_r <= SDM_MAX_EFF_GRID; all values finite and >= 0.  Between grid points the table is interpolated
 * bilinearly (first along the radius of the droplet with the larger multiplicity, every operation rounded),
 * outside the grid it is clamped (R16).  Both arrays are HOST pointers and are copied into the
 * workspace; SYNCHRONOUS.  The table stays until replaced; it is independent of the loaded state. */
#define SDM_MAX_EFF_GRID 64
int sdm_set_efficiency_table(sdm_t *h, int32_t n_r, const double *r_grid_host, const double *E_host);

/* Sharding (cells are independent): this handle holds the slice [base, base + n_sd) of a
 * larger, cell-contiguous GLOBAL state.  The Philox counter of a droplet is its global storage index base + i (i its
 * index in this handle), so a shard loaded with the same seed reproduces the unsharded run exactly: same xi, v, and
 * idx_global = base + idx.  The stable compaction shifts the droplets of later shards, so after every sdm_remove_zero
 * that removed something the caller re-derives each shard's base as the exclusive scan of the shards' survivor counts
 * (paper_2101_06318_b200/sharding.py: rebase).  Default 0.  Stays until changed (sdm_set_state does not reset it).
 * Host-side only (no device work).  Errors: SDM_EINVAL unless 0 <= base and base + capacity <= 2^32 (the counter's
 * index word is 32 bits wide in the kernels). */
int sdm_set_index_base(sdm_t *h, int64_t base);

/* User-supplied kernel code for SDM_KERNEL_USER (the paper keeps the pair logic apart from "potentially user-supplied
 * kernel code"; Fig. 8 runs a second kernel family through the same interface).
 * cuda_src is CUDA C++ source text (host pointer, NUL-terminated) that defines
 *     __device__ double sdm_user_kernel(double vj, double vk, const double *params);
 * returning a(v_j, v_k) [m^3/s] for the pair's volumes, vj being the member with the larger multiplicity (first-in-pair
 * on a tie), exactly what the built-in kernels receive; params points to the n_params (0..SDM_MAX_USER_PARAMS) doubles
 * of params_host, copied into the workspace.  The source is compiled at run time (NVRTC, sm_100a, no FMA contraction:
 * every * and + of the user's code is rounded separately, like the library's own arithmetic) into one module with the
 * library's pair code (Eq. 3-6, Fig. 5); steps with SDM_KERNEL_USER build the permutation with the library's kernels and
 * evaluate every candidate pair through it (no probability screening: the library knows no bound of user code).
 * A user kernel that re-expresses a built-in one reproduces it bit for bit.  The kernel should return a finite value
 * >= 0; a pair whose Eq. 3 value p = a * xi_max * norm is not > 0 (the code returned a negative number or NaN) has no
 * event, gamma_tilde = 0 (R20) -- multiplicities never grow.  +inf is capped by Eq. 4 like any large p.
 * SYNCHRONOUS.  Errors: SDM_EINVAL (NULL
 * source, bad n_params, compilation failed: sdm_last_error holds the compiler log), SDM_ECUDA (NVRTC or the module loader
 * unavailable).  The kernel stays until replaced. */
#define SDM_MAX_USER_PARAMS 16
int sdm_set_kernel_source(sdm_t *h, const char *cuda_src, int32_t n_params, const double *params_host);

/* Replaces the cell ids of the super-droplets currently in storage (cell_id_dev[n_sd], storage order) -- the
 * hook for particle displacement, which the paper performs between coalescence steps and outside this API
 * ("cell_id ... updated before this block"; "multi-dimensional" use).
 * Multiplicities and attributes stay.  Validates 0 <= cell_id < n_cell and re-analyses the layout
 * (cell-contiguous or not, largest cell), which decides the path of the next steps.  SYNCHRONOUS.  Errors:
 * SDM_EINVAL (an id out of range: the state is then unusable), SDM_ESTATE. */
int sdm_set_cell_id(sdm_t *h, const int32_t *cell_id_dev);

/* Copies the current state out in storage order.  Any of the array pointers may be NULL.
 * SYNCHRONOUS (returns n_sd on the host).  The arrays must hold at least n_sd elements (capacity
 * is always enough). */
int sdm_get_state(sdm_t *h, int64_t *n_sd, int64_t *xi_dev, double *v_dev, int32_t *cell_id_dev);
int sdm_get_state_host(sdm_t *h, int64_t *n_sd, int64_t *xi_host, double *v_host,
                       int32_t *cell_id_host);

/* One coalescence step: Fig. 3 steps 1-3.
 *   step 1  per-droplet Philox4x32-10 block (counter = storage index and `step`, key = `seed`),
 *           cell_start table, idx = argsort by (cell_id, key64, storage index)
 *   step 2  for every candidate pair (idx[s+2m], idx[s+2m+1]) of every cell: Eq. 3
 *   step 3  gamma = floor(p) + [u < p - floor(p)], gamma_tilde = min(gamma, floor(xi_j/xi_k)) (Eq. 4),
 *           update of xi and v by Eqs. 5-6 / Fig. 5
 * dt >= 0 [s], dV > 0 [m^3] (one volume for all cells).  n_sd does not change.
 * ASYNCHRONOUS.  Errors: SDM_EINVAL (bad dt, dV, kernel), SDM_ESTATE (no valid state), SDM_ECUDA. */
int sdm_coalescence_step(sdm_t *h, double dt, double dV, const sdm_kernel_t *kernel, uint64_t seed,
                         uint64_t step);

/* sdm_coalescence_step followed by sdm_moments(per_cell = 0) of the post-step state, as one call: on
 * the cell-contiguous path both come out of the same kernel (the state is streamed once).  The
 * state after the call is identical to sdm_coalescence_step's; M0 is exact; M1, M2 equal
 * sdm_moments' up to fp64 summation order (<= 1e-12 relative).  ASYNCHRONOUS. */
int sdm_coalescence_step_moments(sdm_t *h, double dt, double dV, const sdm_kernel_t *kernel,
                                 uint64_t seed, uint64_t step, int64_t *m0_dev, double *m1_dev,
                                 double *m2_dev);

/* Step 0 of Fig. 3: removes super-droplets with xi == 0 by a STABLE
 * compaction of (xi, v, cell_id).  n_sd_out == NULL: ASYNCHRONOUS (n_sd stays on the device);
 * otherwise SYNCHRONOUS and *n_sd_out receives the new count. */
int sdm_remove_zero(sdm_t *h, int64_t *n_sd_out);

/* Moments of the size spectrum, M_k = sum xi * v^k for k = 0, 1, 2 (R13).
 * per_cell == 0: one value each; per_cell != 0: n_cell values each.  M0 is exact (int64); M1, M2
 * are fp64 sums (products rounded as (xi*v) and (xi*v)*v).  ASYNCHRONOUS for _dev outputs;
 * the _host variant is SYNCHRONOUS. */
int sdm_moments(sdm_t *h, int per_cell, int64_t *m0_dev, double *m1_dev, double *m2_dev);
int sdm_moments_host(sdm_t *h, int per_cell, int64_t *m0_host, double *m1_host, double *m2_host);

/* The global moments of sdm_moments(per_cell = 0) for callers that CANNOT allocate device memory -- no handle, no
 * workspace, nothing to create or destroy.  Meant for code that owns (xi, v) on the device but has no way to get
 * scratch memory when it wants the numbers: a host model whose own pool took the whole device at start-up, a
 * monitoring hook on a thread that must not stall the device (cudaMalloc and cudaFree synchronise it), a plug-in in a
 * process whose device-memory budget is fixed.  The partial sums and the arrival counter of the grid-wide reduction
 * live in a static device array inside libsdm itself: SDM_NOALLOC_SCRATCH_BYTES on EVERY GPU that loads the library,
 * held until the process exits.  The call itself performs no cudaMalloc, cudaFree or any other allocating call.
 *   xi_dev[n_sd], v_dev[n_sd]  DEVICE pointers, 16-byte aligned, read only (may be NULL when n_sd == 0)
 *   n_sd                       0 <= n_sd <= SDM_NOALLOC_MAX_SD (the kernels' 32-bit storage indices; the scratch need
 *                              does not grow with n_sd); beyond it: SDM_ECAPACITY and a message naming the limit
 *   m0_dev, m1_dev, m2_dev     DEVICE pointers to one int64 / double / double: M0 exact, M1 and M2 fp64 sums with the
 *                              products rounded as (xi*v) and (xi*v)*v, equal to sdm_moments' to <= 1e-12 relative
 *   cuda_stream                a cudaStream_t of the CURRENT device (NULL = legacy default stream); ASYNCHRONOUS
 *   err_host, err_len          optional HOST buffer for a NUL-terminated message on failure (NULL / 0: none)
 * The pointers and the stream must belong to the device that is current when the call is made.
 * ONE ARRAY PER DEVICE IS SHARED BY ALL CALLS: calls that can overlap on the GPU (two streams, two threads) race on
 * it and return wrong numbers; order them (one stream, or events).  The array keeps the previous call's contents;
 * the call clears what has to start at zero and never reads a partial it did not write itself.
 * The first call on a device looks up the array's device address (cudaGetSymbolAddress) and keeps it: make that first
 * call before any stream capture begins.  Returns SDM_OK, SDM_EINVAL (negative n_sd, NULL or misaligned pointer),
 * SDM_ECAPACITY (n_sd too large), SDM_ECUDA (no device, address look-up or launch failed). */
#define SDM_NOALLOC_MAX_SD 2139095040 /* = SDM_MAX_CAPACITY */
#define SDM_NOALLOC_SCRATCH_BYTES 28672 /* 256 B counter + 1184 CTAs x 3 partials x 8 B */
int sdm_moments_noalloc(const int64_t *xi_dev, const double *v_dev, int64_t n_sd, int64_t *m0_dev, double *m1_dev,
                        double *m2_dev, void *cuda_stream, char *err_host, size_t err_len);

/* The spectrum product of Fig. 6: mass of droplets per unit of ln r [kg per m^3 of air per
 * unit ln r] on n_bins bins (1 <= n_bins <= SDM_MAX_BINS), all cells together.  Bin b holds the droplets with
 * v_edges_host[b] <= v < v_edges_host[b+1] (volumes, strictly increasing, n_bins + 1 values); its value is
 * (sum xi*v) * rho / V / dlnr_host[b], where dlnr_host[b] = ln(r_{b+1} / r_b) > 0 is supplied by the caller
 * (no logarithm is evaluated by the library), rho is the particle density [kg/m^3] and V the volume of air
 * the state represents [m^3]; then n_smooth (>= 0; the paper: 2) passes of a centered five-bin running mean
 * whose window is truncated at the ends (R17).  All array arguments are HOST pointers; out_host
 * receives n_bins values.  SYNCHRONOUS.  The bin sums are fp64 sums in no fixed order (<= 1e-12 relative). */
#define SDM_MAX_BINS 1024
int sdm_spectrum(sdm_t *h, int32_t n_bins, const double *v_edges_host, const double *dlnr_host, double rho,
                 double V, int32_t n_smooth, double *out_host);

/* Exports the permutation and cell table of the LAST sdm_coalescence_step (parity / debugging;
 * the paper's `idx` and `cell_start`): idx_dev[n_sd] (storage indices in
 * cell-major, key-ascending order), cell_start_dev[n_cell + 1].  Either may be NULL.  The copies
 * are enqueued on the stream; with idx_dev != NULL the call first synchronises to learn n_sd. */
int sdm_get_permutation(sdm_t *h, int32_t *idx_dev, int32_t *cell_start_dev);

/* n_steps timesteps [sdm_remove_zero (if remove_zero_each_step); sdm_coalescence_step] with
 * step = step0, step0+1, ...; results equal the per-step calls.  ASYNCHRONOUS.
 *  - A single-cell box (n_cell == 1) with a built-in kernel runs all n_steps in ONE persistent launch.  With
 *    SDM_KERNEL_USER (or when no cooperative grid fits the context) the call is a host loop of per-step launches.
 *  - Shards (sdm_set_index_base): the index base is fixed for the whole call, while a removal in an EARLIER shard
 *    shifts the global storage indices of this one.  With remove_zero_each_step != 0, a sharded run therefore equals
 *    the unsharded run only as long as no earlier shard loses a droplet inside the call; from the first such removal
 *    on it draws other random numbers (still a valid SDM realisation, no longer the same one).  For bit-for-bit
 *    equality use the per-step calls and re-derive the bases after every removal (sharding.py: rebase), or verify
 *    after the call that no shard's n_sd changed (bench.py does). */
int sdm_run(sdm_t *h, double dt, double dV, const sdm_kernel_t *kernel, uint64_t seed,
            uint64_t step0, int64_t n_steps, int remove_zero_each_step);

/* Testing hook for row a3 (the tie rule R7 cannot be reached with Philox output): runs rows a2-a3 of one step on the
 * current state with the CALLER'S 64-bit sort keys, keys_dev[n_sd] by storage index, in place of Philox words 0-1,
 * through the very kernels a real step of this state would use (fused, general or box path, their truncated-key and
 * equal-key branches included); no pair is evaluated and the state does not change.  The result is read with
 * sdm_get_permutation: idx = argsort by (cell_id, key, storage index).  ASYNCHRONOUS. */
int sdm_debug_permutation(sdm_t *h, const uint64_t *keys_dev);

/* Reads SDM_CNT_COUNT counters into counters_host.  SYNCHRONOUS. */
int sdm_get_counters(sdm_t *h, int64_t *counters_host);

/* With SDM_OPT_TIMING on: synchronises, sums the CUDA-event durations [ms] recorded around the
 * dominant kernel of each coalescence step since the last call (the fused per-cell kernel on the
 * cell-contiguous path, the segment-sort kernel on the general path), returns their number, and
 * clears the record.  At most 4096 launches are recorded between two calls. */
int sdm_get_timing(sdm_t *h, double *total_ms, int64_t *n_launches);

/* Message for the last error on this handle (never NULL; "" if none).  h may be NULL: then the
 * message of the last failed sdm_create on this thread. */
const char *sdm_last_error(const sdm_t *h);

/* ABI version of this header: major*1000 + minor. */
int sdm_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SDM_H */
