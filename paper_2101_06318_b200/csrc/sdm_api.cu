// sdm_api.cu -- host side of libsdm: handle, argument checks, workspace carving, kernel launches.
// Implements include/sdm.h.  No device allocation happens here: all device memory is the caller's
// workspace; the only host allocations are the handle and a small pinned read-back block.
#include "../../include/sdm.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <utility>
#include <vector>

#include <cuda_runtime.h>
#include <math_constants.h>

#include "sdm_kernels.cuh"
#include "sdm_fused.cuh"
#include "sdm_fused_count.cuh"
#include "sdm_general.cuh"
#include "sdm_spectrum.cuh"
#include "sdm_box.cuh"

using namespace sdmk;

namespace {

constexpr size_t kAlign = 256;
constexpr int kMinSegCap = 8;

inline size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

struct Layout {
    size_t xi, v, attr, eff, spec, cell, idx, order, cell_start, cell_start2, cell_cnt, cell_bits, bucket_base, bucket_start,
        bucket_cnt, tile_status, scan_status, part0, part1, part2, mom_out, ctrl, box_ctrl, box_queue, total;
    int64_t nb_max, n_tiles, attr_stride, box_stride;
};

Layout make_layout(int64_t cap, int32_t n_cell, int32_t n_attr)
{
    Layout L{};
    L.nb_max = (int64_t)n_cell + cap / 64 + 4096;
    L.n_tiles = (cap + kCompactTile - 1) / kCompactTile;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
    L.xi = take((size_t)cap * 8);
    L.v = take((size_t)cap * 8);
    L.attr_stride = (cap + 31) / 32 * 32;                       // elements between rows of the extra attributes
    L.attr = take((size_t)(n_attr - 1) * (size_t)L.attr_stride * 8);
    L.cell = take((size_t)cap * 4);
    L.idx = take((size_t)cap * 4);
    L.order = take((size_t)cap * 4);
    L.cell_start = take(((size_t)n_cell + 1) * 4);
    L.cell_start2 = take(((size_t)n_cell + 1) * 4);
    L.cell_cnt = take(((size_t)n_cell + 1) * 4);
    L.cell_bits = take(((size_t)n_cell + 1) * 4);
    L.bucket_base = take(((size_t)n_cell + 1) * 4);
    L.bucket_start = take(((size_t)L.nb_max + 1) * 4);
    L.bucket_cnt = take(((size_t)L.nb_max + 1) * 4 * kRankStride);   // rank counters, one per 32-byte sector
    L.tile_status = take((size_t)L.n_tiles * 8);
    L.scan_status = take((size_t)(((int64_t)n_cell + L.nb_max) / 2048 + 4) * 8);
    L.part0 = take((size_t)kMomentPartials * 8);
    L.part1 = take((size_t)kMomentPartials * 8);
    L.part2 = take((size_t)kMomentPartials * 8);
    L.mom_out = take(3 * 8);
    L.ctrl = take(sizeof(Ctrl));
    L.spec = take((size_t)(4 * SDM_MAX_BINS + 1) * 8);          // spectrum: edges, widths, sums, result
    L.eff = take((size_t)(SDM_MAX_EFF_GRID + SDM_MAX_EFF_GRID * SDM_MAX_EFF_GRID) * 8);   // efficiency grid + table
    // single-cell box path (sdm_box.cuh): control block and the double-buffered record queue, 2 x 8 B per droplet
    L.box_stride = 0;
    if (n_cell == 1 && cap <= (int64_t)kBoxMaxCtas * kBoxMeanMax) {
        // fixed-capacity regions: G * (mean + 12 sqrt(mean) + 32) <= cap + 12 sqrt(255 cap) + 32 * 255 records
        L.box_stride = ((int64_t)((double)cap + 12.0 * std::sqrt(255.0 * (double)cap)) + 8192 + 64) / 32 * 32;
        L.box_ctrl = take(sizeof(BoxCtrl));
        L.box_queue = take((size_t)2 * (size_t)L.box_stride * 8);
    }
    L.total = off;
    return L;
}

thread_local std::string g_create_error;

}  // namespace

struct sdm {
    int64_t capacity = 0;
    int32_t n_cell = 0;
    int32_t n_attr = 1;          // extensive attributes per droplet, volume included
    double *attr = nullptr;      // rows 1..n_attr-1
    double *spec = nullptr;      // spectrum scratch: edges [SDM_MAX_BINS+1], dlnr, sums, out [SDM_MAX_BINS each]
    double *eff = nullptr;       // efficiency grid [SDM_MAX_EFF_GRID] followed by the table
    int eff_n = 0;               // 0: no table loaded
    double eff_max = 0.0;        // largest table entry (screening bounds)
    cudaStream_t stream = nullptr;
    unsigned char *ws = nullptr;
    Layout L{};
    // device views into the workspace
    int64_t *xi = nullptr;
    double *v = nullptr;
    int32_t *cell = nullptr;
    int *idx = nullptr, *order = nullptr, *cell_start = nullptr, *cell_start2 = nullptr, *cell_cnt = nullptr,
        *cell_bits = nullptr, *bucket_base = nullptr, *bucket_start = nullptr, *bucket_cnt = nullptr;
    unsigned long long *tile_status = nullptr, *scan_status = nullptr;
    int64_t *part0 = nullptr;
    double *part1 = nullptr, *part2 = nullptr;
    int64_t *mom0 = nullptr;
    double *mom1 = nullptr, *mom2 = nullptr;
    Ctrl *ctrl = nullptr;
    BoxCtrl *box_ctrl = nullptr;                 // single-cell box path (nullptr: not available for this handle)
    unsigned long long *box_queue = nullptr;
    int box_max_ctas = 0;        // co-resident CTAs of k_box_steps on this device
    Ctrl *ctrl_host = nullptr;   // pinned read-back block
    // host knowledge of the state
    bool valid = false;          // a validated state is loaded
    bool stepped = false;        // idx / cell_start hold the permutation of a step
    int64_t n_ub = 0;            // upper bound of n_sd (exact after every synchronous read-back)
    int max_count = 0;           // largest cell at set_state (cells never grow afterwards)
    bool sorted = false;         // cell_id non-decreasing in storage (preserved by compaction)
    int num_sms = 148;
    int device = 0;              // CUDA device of the workspace; every entry point runs with it current
    // options
    bool force_general = false;
    int seg_cap = kWarpCap;      // fused path: largest cell; general path: only when overridden (tests)
    bool seg_cap_set = false;    // SDM_OPT_SEGMENT_CAP given
    bool table_produced = false; // fused path: the last step's kernel wrote the next cell table into cell_start2
    bool tables_ready = false;   // general path: cell_bits / bucket_base / n_seg are valid for this state
    bool split = false;          // general path: some cell is larger than a sort segment
    int n_seg = 0;               // general path: number of sort segments when split
    bool write_idx = true;
    bool screening = true;
    int lanes_per_cell = 0;      // 0: automatic
    int sort_engine = 0;         // 0: automatic, 1: register sorting network, 2: bucket sort
    bool deterministic = false;  // SDM_OPT_DETERMINISTIC: static cell -> warp mapping
    int ctas_per_sm = 0;         // 0: the kernel's own choice (tuning / scaling experiments)
    uint32_t index_base = 0;     // sdm_set_index_base: global storage index of this handle's droplet 0
    int box_ctas_opt = 0;        // SDM_OPT_BOX_CTAS
    int box_region_cap_opt = 0, box_sort_cap_opt = 0;   // SDM_OPT_BOX_REGION_CAP, SDM_OPT_BOX_SORT_CAP (tests)
    bool timing = false;
    std::vector<cudaEvent_t> ev;   // start/stop pairs around the dominant kernel (SDM_OPT_TIMING)
    size_t ev_used = 0;
    int64_t launches = 0;
    std::string err;
};

namespace {

int fail(sdm_t *h, int code, const std::string &msg)
{
    if (h) h->err = msg; else g_create_error = msg;
    return code;
}

int cuda_fail(sdm_t *h, cudaError_t e, const char *what)
{
    return fail(h, SDM_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

// Entry points make the handle's device current for the duration of the call and restore the caller's.
struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) { prev = -1; return; }
        if (prev == dev) prev = -1; else cudaSetDevice(dev);
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};
#define SDM_ENTER(h)                     \
    if (!(h)) return SDM_EINVAL;         \
    DeviceGuard device_guard_((h)->device)

#define SDM_CUDA(h, call)                                         \
    do {                                                          \
        cudaError_t e_ = (call);                                  \
        if (e_ != cudaSuccess) return cuda_fail((h), e_, #call);  \
    } while (0)

#define SDM_LAUNCH(h, kernel, grid, block, smem, ...)                         \
    do {                                                                      \
        kernel<<<(grid), (block), (smem), (h)->stream>>>(__VA_ARGS__);        \
        (h)->launches += 1;                                                   \
        cudaError_t e_ = cudaGetLastError();                                  \
        if (e_ != cudaSuccess) return cuda_fail((h), e_, "launch " #kernel);  \
    } while (0)

constexpr size_t kMaxTimedLaunches = 4096;

// CUDA-event bracket around the dominant kernel (SDM_OPT_TIMING)
int timing_mark(sdm_t *h)
{
    if (!h->timing || h->ev_used >= 2 * kMaxTimedLaunches) return SDM_OK;
    if (h->ev_used >= h->ev.size()) {
        cudaEvent_t e;
        SDM_CUDA(h, cudaEventCreate(&e));
        h->ev.push_back(e);
    }
    SDM_CUDA(h, cudaEventRecord(h->ev[h->ev_used], h->stream));
    h->ev_used += 1;
    return SDM_OK;
}

#define SDM_TIMED(h, stmt)                                 \
    do {                                                   \
        int rc_ = timing_mark(h);                          \
        if (rc_ != SDM_OK) return rc_;                     \
        stmt;                                              \
        rc_ = timing_mark(h);                              \
        if (rc_ != SDM_OK) return rc_;                     \
    } while (0)

inline int grid_for(const sdm_t *h, int64_t work, int block, int per_sm)
{
    int64_t g = (work + block - 1) / block;
    int64_t cap = (int64_t)h->num_sms * per_sm;
    if (g > cap) g = cap;
    if (g < 1) g = 1;
    return (int)g;
}

// single-cell box: persistent cooperative kernel (sdm_box.cuh); number of CTAs for the current droplet count, 0 = not usable
int box_ctas(const sdm_t *h)
{
    if (!h->box_ctrl || h->force_general || h->seg_cap_set || h->box_max_ctas < 1) return 0;
    const int64_t n = h->n_ub > 0 ? h->n_ub : 1;
    int64_t g = (n + 511) / 512;                                // ~512 droplets per CTA for small boxes (measured: C1 best at 16 CTAs)
    if (h->box_ctas_opt > 0) g = h->box_ctas_opt;
    const int64_t cap = std::min<int64_t>(h->box_max_ctas, kBoxMaxCtas);
    if (g > cap) g = cap;
    if (n > g * kBoxMeanMax) return 0;
    return (int)g;
}

bool use_fused(const sdm_t *h)
{
    return h->sorted && !h->force_general && h->max_count <= h->seg_cap && h->max_count <= 512;
}

// [optional remove_zero; step] x n_steps of a single-cell state in one cooperative launch
int enqueue_box(sdm_t *h, const StepParams &prm, int64_t n_steps, int remove_zero)
{
    const int g = box_ctas(h);
    SDM_CUDA(h, cudaMemsetAsync(h->box_ctrl, 0, sizeof(BoxCtrl), h->stream));
    StepParams p = prm;
    while (n_steps > 0) {
        int chunk = (int)std::min<int64_t>(n_steps, 1 << 20);
        long long stride = h->L.box_stride;
        // capacity of a region of the record queue: mean + 12 sigma (+ 32) of a Binomial(n, 1/G) count
        const int64_t mean = (h->n_ub + g - 1) / g;
        int region_cap = (int)(mean + (int64_t)(12.0 * std::sqrt((double)mean)) + 32);
        if ((int64_t)region_cap * g > stride || region_cap > kBoxRegionMax)
            return fail(h, SDM_EINVAL, "internal: box region capacity exceeds the workspace");
        if (h->box_region_cap_opt > 0) region_cap = std::min(region_cap, h->box_region_cap_opt);
        int sort_cap = h->box_sort_cap_opt > 0 ? std::min(h->box_sort_cap_opt, kBoxRegionMax) : kBoxRegionMax;
        void *args[] = {&h->xi, &h->v, &h->cell, &h->idx, &h->cell_start, &h->ctrl, &h->box_ctrl, &h->box_queue, &stride,
                        &region_cap, &sort_cap, &h->tile_status, &chunk, &remove_zero, &p};
        cudaError_t e = cudaLaunchCooperativeKernel((const void *)k_box_steps, dim3(g), dim3(kBoxThreads), args, kBoxSmemBytes,
                                                    h->stream);
        h->launches += 1;
        if (e != cudaSuccess) return cuda_fail(h, e, "launch k_box_steps");
        n_steps -= chunk;
        if (n_steps > 0) {
            SDM_CUDA(h, cudaMemsetAsync(h->box_ctrl, 0, sizeof(BoxCtrl), h->stream));
            p.step += (uint64_t)chunk;
        }
    }
    return SDM_OK;
}

// largest segment of the general path: the warp counting sort holds 256 droplets
int general_cap(const sdm_t *h) { return h->seg_cap_set ? h->seg_cap : kGenCap; }


AttrView attr_view(const sdm_t *h)
{
    AttrView av{};
    av.p = h->attr;
    av.stride = h->L.attr_stride;
    av.n = h->n_attr - 1;
    av.eff_n = h->eff_n;
    av.eff_grid = h->eff;
    av.eff_tab = h->eff + SDM_MAX_EFF_GRID;
    return av;
}

int read_ctrl(sdm_t *h)
{
    SDM_CUDA(h, cudaMemcpyAsync(h->ctrl_host, h->ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, h->stream));
    SDM_CUDA(h, cudaStreamSynchronize(h->stream));
    return SDM_OK;
}

int make_params(sdm_t *h, double dt, double dV, const sdm_kernel_t *kernel, uint64_t seed,
                uint64_t step, StepParams &prm)
{
    if (!kernel) return fail(h, SDM_EINVAL, "kernel is NULL");
    if (!(dt >= 0.0) || !(dV > 0.0) || !std::isfinite(dt) || !std::isfinite(dV))
        return fail(h, SDM_EINVAL, "need dt >= 0 and dV > 0, both finite");
    if (kernel->type != SDM_KERNEL_GOLOVIN && kernel->type != SDM_KERNEL_GRAVITATIONAL &&
        kernel->type != SDM_KERNEL_GRAVITATIONAL_TABULATED)
        return fail(h, SDM_EINVAL, "unknown kernel type");
    if (kernel->type == SDM_KERNEL_GRAVITATIONAL_TABULATED && h->eff_n < 2)
        return fail(h, SDM_EINVAL, "SDM_KERNEL_GRAVITATIONAL_TABULATED needs sdm_set_efficiency_table first");
    if (kernel->reserved != 0) return fail(h, SDM_EINVAL, "kernel.reserved must be 0");
    double kp = kernel->type == SDM_KERNEL_GOLOVIN ? kernel->b : kernel->E;
    if (!std::isfinite(kp) || kp < 0.0) return fail(h, SDM_EINVAL, "kernel parameter must be finite and >= 0");
    prm = StepParams{};
    prm.dtdv = dt / dV;
    prm.kparam = kp;
    prm.kparam_ub = kernel->type == SDM_KERNEL_GRAVITATIONAL_TABULATED ? kp * h->eff_max : kp;
    prm.kernel = kernel->type;
    prm.write_idx = h->write_idx ? 1 : 0;
    prm.seed = seed;
    prm.step = step;
    prm.screening = h->screening ? 1 : 0;
    prm.attr = attr_view(h);
    auto float_ru = [](double x) {                      // smallest fp32 >= x (inf stays inf)
        float f = (float)x;
        if ((double)f < x) f = std::nextafterf(f, INFINITY);
        return f;
    };
    prm.dtdv_ub_f = float_ru(prm.dtdv);
    prm.kparam_ub_f = float_ru(prm.kparam_ub);
    philox_round_keys(seed, h->index_base, prm.rk);
    return SDM_OK;
}

// General path: the static split of large cells into sort segments (cell_bits, bucket_base, n_seg), decided
// from the current cell counts; SYNCHRONOUS (reads n_seg back), done once per loaded state / option change.
int build_tables(sdm_t *h)
{
    const int gcap = general_cap(h);
    h->split = h->max_count > gcap;
    SDM_LAUNCH(h, k_cell_count, h->n_cell <= kCellCountBins ? grid_for(h, h->n_ub, 256, 4) : grid_for(h, h->n_ub, 256, 16),
               256, 0, h->cell, h->ctrl, h->n_cell, h->cell_cnt);
    SDM_LAUNCH(h, k_cell_scan, 1, kScanThreads, 0, h->cell_cnt, h->n_cell, h->cell_start, h->split ? 1 : 0, gcap,
               h->cell_bits, h->bucket_base, h->ctrl);
    int rc = read_ctrl(h);
    if (rc != SDM_OK) return rc;
    h->n_seg = h->ctrl_host->n_buckets;
    if (h->n_seg > h->L.nb_max) return fail(h, SDM_EINVAL, "segment table exceeds the workspace (segment cap too small)");
    h->tables_ready = true;
    return SDM_OK;
}

// Fig. 3 steps 1-3 enqueued on the stream
int enqueue_moments(sdm_t *h, int per_cell, int64_t *m0, double *m1, double *m2);

// m0/m1/m2 != NULL: also produce the global moments of the post-step state
int enqueue_step(sdm_t *h, const StepParams &prm, int64_t *m0 = nullptr, double *m1 = nullptr,
                 double *m2 = nullptr)
{
    const int64_t n_ub = h->n_ub;
    const bool produced = h->table_produced;      // did the previous step's kernel leave the next cell table?
    h->table_produced = false;
    if (box_ctas(h) > 0) {
        SDM_TIMED(h, { int rc_box = enqueue_box(h, prm, 1, 0); if (rc_box != SDM_OK) return rc_box; });
        if (m0) return enqueue_moments(h, 0, m0, m1, m2);
        return SDM_OK;
    }
    if (use_fused(h)) {
        // row a2: the counting-sort kernel derives the NEXT step's table from cell_id while it runs (written
        // to cell_start2); when it did so last step, k_cell_start_sorted only rebuilds the table if a
        // compaction has moved droplets since (device flag), else it returns at once
        if (produced) std::swap(h->cell_start, h->cell_start2);
        const int gb_count = grid_for(h, (int64_t)h->n_cell * 32, kCountWarps * 32,
                                      h->ctas_per_sm > 0 ? h->ctas_per_sm : kCountBlocksPerSM);
        SDM_LAUNCH(h, k_cell_start_sorted, grid_for(h, (n_ub + 4 * kCellStartQuads - 1) / (4 * kCellStartQuads), 256, 8), 256, 0, h->cell, h->ctrl, h->n_cell,
                   h->cell_start, produced ? 0 : 1, gb_count * kCountWarps);
        // shape of the per-cell kernel: E droplets per lane, L lanes per cell (capacity E*L).  Eight
        // droplets per lane keep the unrolled network inside the instruction cache; wider shapes lose
        // more to instruction fetch than they save in shuffles (measured).
        const bool bucket = h->max_count <= kCountCap &&
                            (h->sort_engine == 2 || (h->sort_engine == 0 && h->max_count > 128));
        if (bucket) {
            const int gb = gb_count;
            if (m0 && gb > kMomentPartials) return fail(h, SDM_EINVAL, "grid exceeds the moment partials (lower SDM_OPT_CTAS_PER_SM)");
#define SDM_COUNT_K(MM, TT, KK)                                                                                   \
    SDM_TIMED(h, SDM_LAUNCH(h, (k_fused_cells_count<MM, TT, KK>), gb, kCountWarps * 32, kCountSmemBytes, h->xi, h->v,   \
                            h->cell, h->cell_start, h->cell_start2, h->n_cell, h->idx, h->ctrl, prm, h->part0,        \
                            h->part1, h->part2, m0, m1, m2))
#define SDM_COUNT(MM, TT)                                                                                         \
    do {                                                                                                          \
        if (tickets) SDM_COUNT_K(MM, TT, true);                                                                   \
        else SDM_COUNT_K(MM, TT, false);                                                                          \
    } while (0)
            const bool tab = prm.kernel == SDM_KERNEL_GRAVITATIONAL_TABULATED;
            // chunk tickets pay off when a warp gets many chunks; small tables keep the static stride
            const bool tickets = !h->deterministic && (int64_t)h->n_cell >= (int64_t)32 * gb * kCountWarps;
            if (m0 && tab) SDM_COUNT(true, true);
            else if (m0) SDM_COUNT(true, false);
            else if (tab) SDM_COUNT(false, true);
            else SDM_COUNT(false, false);
#undef SDM_COUNT_K
#undef SDM_COUNT
            h->table_produced = true;
            return SDM_OK;
        }
        int E = 8, L = 8;
        if (h->max_count > 256) { E = 16; L = 32; }
        else if (h->max_count > 128) { E = 8; L = 32; }
        else if (h->max_count > 64) { E = 8; L = 16; }
        if (h->lanes_per_cell == 16 && h->max_count > 128 && h->max_count <= 256) { E = 16; L = 16; }
        const int64_t warps_needed = ((int64_t)h->n_cell * L + 31) / 32;
        const int gf = std::min(grid_for(h, warps_needed * 32, kFusedWarps * 32, 8), kMomentPartials);
#define SDM_FUSED_T(EE, LL, MM, TT)                                                                          \
    SDM_TIMED(h, SDM_LAUNCH(h, (k_fused_cells<EE, LL, MM, TT>), gf, kFusedWarps * 32, 0, h->xi, h->v,            \
                            h->cell_start, h->n_cell, h->idx, h->ctrl, prm, h->part0, h->part1, h->part2, m0,    \
                            m1, m2))
#define SDM_FUSED(EE, LL)                                                                                    \
    do {                                                                                                     \
        const bool tab_ = prm.kernel == SDM_KERNEL_GRAVITATIONAL_TABULATED;                                  \
        if (m0 && tab_) SDM_FUSED_T(EE, LL, true, true);                                                     \
        else if (m0) SDM_FUSED_T(EE, LL, true, false);                                                       \
        else if (tab_) SDM_FUSED_T(EE, LL, false, true);                                                     \
        else SDM_FUSED_T(EE, LL, false, false);                                                              \
    } while (0)
        if (E == 8 && L == 8) SDM_FUSED(8, 8);
        else if (E == 8 && L == 16) SDM_FUSED(8, 16);
        else if (E == 8 && L == 32) SDM_FUSED(8, 32);
        else if (E == 16 && L == 16) SDM_FUSED(16, 16);
        else SDM_FUSED(16, 32);
#undef SDM_FUSED
#undef SDM_FUSED_T
        return SDM_OK;
    }
    if (!h->tables_ready) {
        int rc = build_tables(h);
        if (rc != SDM_OK) return rc;
    }
    const int split = h->split ? 1 : 0;
    const int n_seg = split ? h->n_seg : h->n_cell;
    int *seg_start = split ? h->bucket_start : h->cell_start;
    const int g = grid_for(h, n_ub, 256, 16);
    // idx[] carries the arrival ranks from the count to the scatter pass; the sort kernel overwrites it afterwards
    SDM_LAUNCH(h, k_gen_count, (split && h->n_cell <= kCellCountBins) ? grid_for(h, n_ub, 256, 8) : g, 256, 0, h->cell,
               h->ctrl, h->n_cell, split, h->cell_bits, h->bucket_base, h->cell_cnt, h->bucket_cnt, h->idx, prm);
    const int scan_tiles = (h->n_cell + kScanTile - 1) / kScanTile + (split ? (n_seg + kScanTile - 1) / kScanTile : 0);
    SDM_LAUNCH(h, k_gen_scan, scan_tiles < 4 * h->num_sms ? scan_tiles : 4 * h->num_sms, kScanTileThreads, 0, split ? h->cell_cnt : h->bucket_cnt,
               split ? 1 : kRankStride, h->n_cell, h->cell_start, split, h->bucket_cnt, kRankStride, n_seg,
               h->bucket_start, h->ctrl, h->scan_status);
    SDM_LAUNCH(h, k_gen_scatter, g, 256, 0, h->cell, h->ctrl, split, h->cell_bits, h->bucket_base, seg_start,
               h->idx, h->order, prm);
    // four droplets per lane when no segment can exceed 128 (half the Philox blocks per warp), else eight
    if ((split ? general_cap(h) : h->max_count) <= 128)
        SDM_TIMED(h, SDM_LAUNCH(h, k_segment_sort_pairs<4>, grid_for(h, (int64_t)n_seg * 32, kGenWarps * 32, 4),
                                kGenWarps * 32, kGenSmemBytes, seg_start, n_seg, split, general_cap(h), h->order,
                                h->cell, h->cell_bits, h->cell_start, h->idx, h->xi, h->v, h->ctrl, prm));
    else
        SDM_TIMED(h, SDM_LAUNCH(h, k_segment_sort_pairs<8>, grid_for(h, (int64_t)n_seg * 32, kGenWarps * 32, 4),
                                kGenWarps * 32, kGenSmemBytes, seg_start, n_seg, split, general_cap(h), h->order,
                                h->cell, h->cell_bits, h->cell_start, h->idx, h->xi, h->v, h->ctrl, prm));
    if (split)
        SDM_LAUNCH(h, k_pairs_straddle, grid_for(h, n_seg, 256, 8), 256, 0, seg_start, n_seg, h->idx, h->cell,
                   h->cell_start, h->xi, h->v, h->ctrl, prm);
    if (m0) return enqueue_moments(h, 0, m0, m1, m2);
    return SDM_OK;
}

int enqueue_remove_zero(sdm_t *h)
{
    int64_t tiles = (h->n_ub + kCompactTile - 1) / kCompactTile;
    SDM_LAUNCH(h, k_compact, grid_for(h, tiles * kCompactThreads, kCompactThreads, 4), kCompactThreads,
               (size_t)(h->n_attr - 1) * kCompactTile * 8, h->xi, h->v, h->cell, h->ctrl, h->tile_status, attr_view(h));
    h->stepped = false;                       // idx no longer refers to the current storage order
    return SDM_OK;
}

int enqueue_moments(sdm_t *h, int per_cell, int64_t *m0, double *m1, double *m2)
{
    if (!per_cell) {
        // small states: fewer CTAs (the last CTA sums one partial per CTA)
        int64_t mb = (h->n_ub / 2 + (int64_t)kMomentThreads * 4 - 1) / ((int64_t)kMomentThreads * 4);
        mb = mb < 1 ? 1 : (mb > kMomentBlocks ? kMomentBlocks : mb);
        SDM_LAUNCH(h, k_moments_global, (int)mb, kMomentThreads, 0, h->xi, h->v, h->ctrl, h->part0,
                   h->part1, h->part2, m0, m1, m2);
        return SDM_OK;
    }
    SDM_LAUNCH(h, k_moments_zero, grid_for(h, h->n_cell, 256, 8), 256, 0, h->n_cell, m0, m1, m2);
    SDM_LAUNCH(h, k_moments_cell_atomic, grid_for(h, h->n_ub, 256, 16), 256, 0, h->xi, h->v, h->cell,
               h->ctrl, m0, m1, m2);
    return SDM_OK;
}

int load_state_common(sdm_t *h, int64_t n_sd)
{
    // validation + layout analysis; synchronous
    Ctrl zero{};
    zero.n = (int)n_sd;
    zero.epoch = 1;                                   // tile status words are tagged; 0 = never written
    zero.scan_epoch = 1;
    SDM_CUDA(h, cudaMemsetAsync(h->tile_status, 0, (size_t)h->L.n_tiles * 8, h->stream));
    SDM_CUDA(h, cudaMemsetAsync(h->scan_status, 0, (size_t)(((int64_t)h->n_cell + h->L.nb_max) / 2048 + 4) * 8, h->stream));
    if (h->n_attr > 1)
        SDM_CUDA(h, cudaMemsetAsync(h->attr, 0, (size_t)(h->n_attr - 1) * (size_t)h->L.attr_stride * 8, h->stream));
    SDM_CUDA(h, cudaMemcpyAsync(h->ctrl, &zero, sizeof(Ctrl), cudaMemcpyHostToDevice, h->stream));
    SDM_CUDA(h, cudaStreamSynchronize(h->stream));   // `zero` lives on this stack frame
    SDM_CUDA(h, cudaMemsetAsync(h->cell_cnt, 0, ((size_t)h->n_cell + 1) * 4, h->stream));
    if (n_sd > 0)
        SDM_LAUNCH(h, k_analyze, grid_for(h, n_sd, 256, 16), 256, 0, h->xi, h->v, h->cell, (int)n_sd, h->n_cell,
                   h->cell_cnt, h->ctrl);
    SDM_LAUNCH(h, k_max_count, grid_for(h, h->n_cell, 256, 8), 256, 0, h->cell_cnt, h->n_cell, h->ctrl);
    int rc = read_ctrl(h);
    if (rc != SDM_OK) return rc;
    h->stepped = false;
    if (h->ctrl_host->invalid) {
        h->valid = false;
        return fail(h, SDM_EINVAL,
                    "state validation failed: need 0 <= cell_id < n_cell, xi >= 0, v finite and > 0");
    }
    h->valid = true;
    h->table_produced = false;
    h->tables_ready = false;
    h->n_ub = n_sd;
    h->max_count = h->ctrl_host->max_count;
    h->sorted = (h->ctrl_host->unsorted == 0);
    return SDM_OK;
}

}  // namespace

extern "C" {

int sdm_version(void) { return 2000; }

size_t sdm_workspace_bytes_attr(int64_t capacity, int32_t n_cell, int32_t n_attr)
{
    if (capacity < 1 || capacity > (int64_t)SDM_MAX_CAPACITY || n_cell < 1 || n_attr < 1 || n_attr > SDM_MAX_ATTR)
        return 0;
    return make_layout(capacity, n_cell, n_attr).total;
}

size_t sdm_workspace_bytes(int64_t capacity, int32_t n_cell) { return sdm_workspace_bytes_attr(capacity, n_cell, 1); }

const char *sdm_last_error(const sdm_t *h) { return h ? h->err.c_str() : g_create_error.c_str(); }

int sdm_create(sdm_t **out, int64_t capacity, int32_t n_cell, void *workspace_dev, size_t workspace_bytes,
               void *cuda_stream)
{
    return sdm_create_attr(out, capacity, n_cell, 1, workspace_dev, workspace_bytes, cuda_stream);
}

int sdm_create_attr(sdm_t **out, int64_t capacity, int32_t n_cell, int32_t n_attr, void *workspace_dev,
                    size_t workspace_bytes, void *cuda_stream)
{
    if (!out) return fail(nullptr, SDM_EINVAL, "out is NULL");
    *out = nullptr;
    size_t need = sdm_workspace_bytes_attr(capacity, n_cell, n_attr);
    if (need == 0) return fail(nullptr, SDM_EINVAL, "invalid capacity, n_cell or n_attr");
    if (!workspace_dev) return fail(nullptr, SDM_EINVAL, "workspace is NULL");
    if (reinterpret_cast<uintptr_t>(workspace_dev) % kAlign != 0)
        return fail(nullptr, SDM_EINVAL, "workspace must be 256-byte aligned");
    if (workspace_bytes < need) return fail(nullptr, SDM_EINVAL, "workspace too small (see sdm_workspace_bytes)");
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetDevice (no CUDA device? there is no CPU fallback)");
    cudaPointerAttributes pa{};                           // the handle lives on the device that owns the workspace
    if (cudaPointerGetAttributes(&pa, workspace_dev) == cudaSuccess && pa.type == cudaMemoryTypeDevice) dev = pa.device;
    else cudaGetLastError();
    DeviceGuard device_guard_(dev);
    cudaDeviceProp prop{};
    e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetDeviceProperties");
    sdm_t *h = new (std::nothrow) sdm();
    if (!h) return fail(nullptr, SDM_EINVAL, "out of host memory");
    h->capacity = capacity;
    h->n_cell = n_cell;
    h->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    h->ws = static_cast<unsigned char *>(workspace_dev);
    h->n_attr = n_attr;
    h->L = make_layout(capacity, n_cell, n_attr);
    h->num_sms = prop.multiProcessorCount > 0 ? prop.multiProcessorCount : 148;
    h->device = dev;
    const Layout &L = h->L;
    h->xi = reinterpret_cast<int64_t *>(h->ws + L.xi);
    h->v = reinterpret_cast<double *>(h->ws + L.v);
    h->attr = reinterpret_cast<double *>(h->ws + L.attr);
    h->eff = reinterpret_cast<double *>(h->ws + L.eff);
    h->spec = reinterpret_cast<double *>(h->ws + L.spec);
    h->cell = reinterpret_cast<int32_t *>(h->ws + L.cell);
    h->idx = reinterpret_cast<int *>(h->ws + L.idx);
    h->order = reinterpret_cast<int *>(h->ws + L.order);
    h->cell_start = reinterpret_cast<int *>(h->ws + L.cell_start);
    h->cell_start2 = reinterpret_cast<int *>(h->ws + L.cell_start2);
    h->cell_cnt = reinterpret_cast<int *>(h->ws + L.cell_cnt);
    h->cell_bits = reinterpret_cast<int *>(h->ws + L.cell_bits);
    h->bucket_base = reinterpret_cast<int *>(h->ws + L.bucket_base);
    h->bucket_start = reinterpret_cast<int *>(h->ws + L.bucket_start);
    h->bucket_cnt = reinterpret_cast<int *>(h->ws + L.bucket_cnt);
    h->tile_status = reinterpret_cast<unsigned long long *>(h->ws + L.tile_status);
    h->scan_status = reinterpret_cast<unsigned long long *>(h->ws + L.scan_status);
    h->part0 = reinterpret_cast<int64_t *>(h->ws + L.part0);
    h->part1 = reinterpret_cast<double *>(h->ws + L.part1);
    h->part2 = reinterpret_cast<double *>(h->ws + L.part2);
    h->mom0 = reinterpret_cast<int64_t *>(h->ws + L.mom_out);
    h->mom1 = reinterpret_cast<double *>(h->ws + L.mom_out + 8);
    h->mom2 = reinterpret_cast<double *>(h->ws + L.mom_out + 16);
    h->ctrl = reinterpret_cast<Ctrl *>(h->ws + L.ctrl);
    if (L.box_stride > 0) {
        h->box_ctrl = reinterpret_cast<BoxCtrl *>(h->ws + L.box_ctrl);
        h->box_queue = reinterpret_cast<unsigned long long *>(h->ws + L.box_queue);
    }
    auto bail = [&](cudaError_t ce, const char *what) {
        int rc = cuda_fail(nullptr, ce, what);
        if (h->ctrl_host) cudaFreeHost(h->ctrl_host);
        delete h;
        return rc;
    };
    e = cudaMallocHost(reinterpret_cast<void **>(&h->ctrl_host), sizeof(Ctrl));
    if (e != cudaSuccess) { h->ctrl_host = nullptr; return bail(e, "cudaMallocHost"); }
    e = cudaFuncSetAttribute(k_segment_sort_pairs<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kGenSmemBytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_segment_sort_pairs<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kGenSmemBytes);
    if (e != cudaSuccess) return bail(e, "cudaFuncSetAttribute(k_segment_sort_pairs)");
    e = cudaSuccess;
#define SDM_SMEM_ATTR(MM, TT, KK)                                                                              \
    if (e == cudaSuccess)                                                                                      \
        e = cudaFuncSetAttribute(k_fused_cells_count<MM, TT, KK>, cudaFuncAttributeMaxDynamicSharedMemorySize,   \
                                 (int)kCountSmemBytes)
    SDM_SMEM_ATTR(true, false, true); SDM_SMEM_ATTR(false, false, true);
    SDM_SMEM_ATTR(true, true, true); SDM_SMEM_ATTR(false, true, true);
    SDM_SMEM_ATTR(true, false, false); SDM_SMEM_ATTR(false, false, false);
    SDM_SMEM_ATTR(true, true, false); SDM_SMEM_ATTR(false, true, false);
#undef SDM_SMEM_ATTR
    if (e != cudaSuccess) return bail(e, "cudaFuncSetAttribute(k_fused_cells_count)");
    if (h->box_ctrl) {
        int coop = 0, per_sm = 0;
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
        e = cudaFuncSetAttribute(k_box_steps, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kBoxSmemBytes);
        if (e == cudaSuccess)
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_box_steps, kBoxThreads, kBoxSmemBytes);
        if (e != cudaSuccess) return bail(e, "k_box_steps attributes");
        h->box_max_ctas = coop ? per_sm * h->num_sms : 0;
    }
    if (n_attr > 1) {
        e = cudaFuncSetAttribute(k_compact, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)((SDM_MAX_ATTR - 1) * kCompactTile * 8));
        if (e != cudaSuccess) return bail(e, "cudaFuncSetAttribute(k_compact)");
    }
    e = cudaMemsetAsync(h->ctrl, 0, sizeof(Ctrl), h->stream);
    if (e != cudaSuccess) return bail(e, "cudaMemsetAsync(ctrl)");
    e = cudaMemsetAsync(h->spec, 0, (size_t)(4 * SDM_MAX_BINS + 1) * 8, h->stream);
    if (e != cudaSuccess) return bail(e, "cudaMemsetAsync(spec)");
    e = cudaMemsetAsync(h->cell_cnt, 0, ((size_t)n_cell + 1) * 4, h->stream);
    if (e != cudaSuccess) return bail(e, "cudaMemsetAsync(cell_cnt)");
    e = cudaMemsetAsync(h->bucket_cnt, 0, ((size_t)h->L.nb_max + 1) * 4 * kRankStride, h->stream);
    if (e != cudaSuccess) return bail(e, "cudaMemsetAsync(bucket_cnt)");
    e = cudaMemsetAsync(h->cell_start, 0, ((size_t)n_cell + 1) * 4, h->stream);
    if (e != cudaSuccess) return bail(e, "cudaMemsetAsync(cell_start)");
    e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return bail(e, "cudaStreamSynchronize");
    *out = h;
    return SDM_OK;
}

int sdm_destroy(sdm_t *h)
{
    SDM_ENTER(h);
    cudaStreamSynchronize(h->stream);
    if (h->ctrl_host) cudaFreeHost(h->ctrl_host);
    for (cudaEvent_t e : h->ev) cudaEventDestroy(e);
    delete h;
    return SDM_OK;
}

int sdm_set_option(sdm_t *h, int32_t option, int64_t value)
{
    SDM_ENTER(h);
    switch (option) {
    case SDM_OPT_FORCE_GENERAL: h->force_general = value != 0; h->tables_ready = false; return SDM_OK;
    case SDM_OPT_SEGMENT_CAP:
        h->tables_ready = false;
        if (value == 0) { h->seg_cap = kWarpCap; h->seg_cap_set = false; return SDM_OK; }
        if (value < kMinSegCap || value > kGenCap) return fail(h, SDM_EINVAL, "segment cap must be in [8, 256]");
        if ((int64_t)h->n_cell + 4 * h->capacity / value + 2 > h->L.nb_max)
            return fail(h, SDM_EINVAL, "segment cap too small for this workspace");
        h->seg_cap = (int)value;
        h->seg_cap_set = true;
        return SDM_OK;
    case SDM_OPT_WRITE_IDX: h->write_idx = value != 0; return SDM_OK;
    case SDM_OPT_SCREENING: h->screening = value != 0; return SDM_OK;
    case SDM_OPT_TIMING: h->timing = value != 0; h->ev_used = 0; return SDM_OK;
    case SDM_OPT_LANES_PER_CELL:
        if (value != 0 && value != 16) return fail(h, SDM_EINVAL, "lanes per cell: 0 or 16");
        h->lanes_per_cell = (int)value;
        return SDM_OK;
    case SDM_OPT_SORT_ENGINE:
        if (value < 0 || value > 2) return fail(h, SDM_EINVAL, "sort engine: 0 (auto), 1 (network) or 2 (bucket)");
        h->sort_engine = (int)value;
        return SDM_OK;
    case SDM_OPT_DETERMINISTIC: h->deterministic = value != 0; return SDM_OK;
    case SDM_OPT_BOX_REGION_CAP:
        if (value < 0 || value > kBoxRegionMax) return fail(h, SDM_EINVAL, "box region capacity: 0 (automatic) .. 9216");
        h->box_region_cap_opt = (int)value;
        return SDM_OK;
    case SDM_OPT_BOX_SORT_CAP:
        if (value < 0 || value > kBoxRegionMax) return fail(h, SDM_EINVAL, "box sort capacity: 0 (automatic) .. 9216");
        h->box_sort_cap_opt = (int)value;
        return SDM_OK;
    case SDM_OPT_BOX_CTAS:
        if (value < 0 || value > kBoxMaxCtas) return fail(h, SDM_EINVAL, "box CTAs: 0 (automatic) .. 255");
        h->box_ctas_opt = (int)value;
        return SDM_OK;
    case SDM_OPT_CTAS_PER_SM:
        if (value < 0 || value > 32) return fail(h, SDM_EINVAL, "CTAs per SM: 0 (automatic) .. 32");
        h->ctas_per_sm = (int)value;
        return SDM_OK;
    default: return fail(h, SDM_EINVAL, "unknown option");
    }
}

int sdm_set_state(sdm_t *h, int64_t n_sd, const int64_t *xi_dev, const double *v_dev, const int32_t *cell_id_dev)
{
    SDM_ENTER(h);
    if (n_sd < 0) return fail(h, SDM_EINVAL, "n_sd < 0");
    if (n_sd > h->capacity) return fail(h, SDM_ECAPACITY, "n_sd exceeds the capacity given to sdm_create");
    if (n_sd > 0 && (!xi_dev || !v_dev || !cell_id_dev)) return fail(h, SDM_EINVAL, "state pointer is NULL");
    h->valid = false;
    if (n_sd > 0) {
        SDM_CUDA(h, cudaMemcpyAsync(h->xi, xi_dev, (size_t)n_sd * 8, cudaMemcpyDeviceToDevice, h->stream));
        SDM_CUDA(h, cudaMemcpyAsync(h->v, v_dev, (size_t)n_sd * 8, cudaMemcpyDeviceToDevice, h->stream));
        SDM_CUDA(h, cudaMemcpyAsync(h->cell, cell_id_dev, (size_t)n_sd * 4, cudaMemcpyDeviceToDevice, h->stream));
    }
    return load_state_common(h, n_sd);
}

int sdm_set_state_host(sdm_t *h, int64_t n_sd, const int64_t *xi_host, const double *v_host,
                       const int32_t *cell_id_host)
{
    SDM_ENTER(h);
    if (n_sd < 0) return fail(h, SDM_EINVAL, "n_sd < 0");
    if (n_sd > h->capacity) return fail(h, SDM_ECAPACITY, "n_sd exceeds the capacity given to sdm_create");
    if (n_sd > 0 && (!xi_host || !v_host || !cell_id_host)) return fail(h, SDM_EINVAL, "state pointer is NULL");
    h->valid = false;
    if (n_sd > 0) {
        SDM_CUDA(h, cudaMemcpyAsync(h->xi, xi_host, (size_t)n_sd * 8, cudaMemcpyHostToDevice, h->stream));
        SDM_CUDA(h, cudaMemcpyAsync(h->v, v_host, (size_t)n_sd * 8, cudaMemcpyHostToDevice, h->stream));
        SDM_CUDA(h, cudaMemcpyAsync(h->cell, cell_id_host, (size_t)n_sd * 4, cudaMemcpyHostToDevice, h->stream));
    }
    return load_state_common(h, n_sd);
}

int sdm_set_index_base(sdm_t *h, int64_t base)
{
    SDM_ENTER(h);
    if (base < 0 || base + h->capacity > ((int64_t)1 << 32))
        return fail(h, SDM_EINVAL, "index base: need 0 <= base and base + capacity <= 2^32");
    h->index_base = (uint32_t)base;
    return SDM_OK;
}

int sdm_set_cell_id(sdm_t *h, const int32_t *cell_id_dev)
{
    SDM_ENTER(h);
    if (!h->valid) return fail(h, SDM_ESTATE, "no valid state loaded");
    int rc = read_ctrl(h);
    if (rc != SDM_OK) return rc;
    const int64_t n = h->ctrl_host->n;
    h->n_ub = n;
    if (n > 0 && !cell_id_dev) return fail(h, SDM_EINVAL, "cell id pointer is NULL");
    h->stepped = false;
    h->table_produced = false;
    h->tables_ready = false;
    if (n > 0) SDM_CUDA(h, cudaMemcpyAsync(h->cell, cell_id_dev, (size_t)n * 4, cudaMemcpyDeviceToDevice, h->stream));
    // reset the layout fields of the control block (cell_cnt[] is all zero between calls)
    SDM_CUDA(h, cudaMemsetAsync(&h->ctrl->unsorted, 0, sizeof(int), h->stream));
    SDM_CUDA(h, cudaMemsetAsync(&h->ctrl->max_count, 0, sizeof(int), h->stream));
    if (n > 0)
        SDM_LAUNCH(h, k_analyze_cells, grid_for(h, n, 256, 16), 256, 0, h->cell, (int)n, h->n_cell, h->cell_cnt, h->ctrl);
    SDM_LAUNCH(h, k_max_count, grid_for(h, h->n_cell, 256, 8), 256, 0, h->cell_cnt, h->n_cell, h->ctrl);
    rc = read_ctrl(h);
    if (rc != SDM_OK) return rc;
    if (h->ctrl_host->invalid) {
        h->valid = false;
        return fail(h, SDM_EINVAL, "cell id validation failed: need 0 <= cell_id < n_cell");
    }
    h->max_count = h->ctrl_host->max_count;
    h->sorted = (h->ctrl_host->unsorted == 0);
    return SDM_OK;
}

int sdm_set_efficiency_table(sdm_t *h, int32_t n_r, const double *r_grid_host, const double *E_host)
{
    SDM_ENTER(h);
    if (n_r < 2 || n_r > SDM_MAX_EFF_GRID) return fail(h, SDM_EINVAL, "need 2 <= n_r <= SDM_MAX_EFF_GRID");
    if (!r_grid_host || !E_host) return fail(h, SDM_EINVAL, "table pointer is NULL");
    for (int i = 0; i < n_r; ++i) {
        if (!(r_grid_host[i] > 0.0) || !std::isfinite(r_grid_host[i]) || (i > 0 && !(r_grid_host[i] > r_grid_host[i - 1])))
            return fail(h, SDM_EINVAL, "radius grid must be positive, finite and strictly increasing");
    }
    double emax = 0.0;
    for (int i = 0; i < n_r * n_r; ++i) {
        if (!(E_host[i] >= 0.0) || !std::isfinite(E_host[i])) return fail(h, SDM_EINVAL, "efficiencies must be finite and >= 0");
        emax = std::fmax(emax, E_host[i]);
    }
    SDM_CUDA(h, cudaStreamSynchronize(h->stream));      // steps that still read the old table
    SDM_CUDA(h, cudaMemcpyAsync(h->eff, r_grid_host, (size_t)n_r * 8, cudaMemcpyHostToDevice, h->stream));
    SDM_CUDA(h, cudaMemcpyAsync(h->eff + SDM_MAX_EFF_GRID, E_host, (size_t)n_r * n_r * 8, cudaMemcpyHostToDevice, h->stream));
    SDM_CUDA(h, cudaStreamSynchronize(h->stream));
    h->eff_n = n_r;
    h->eff_max = emax;
    return SDM_OK;
}

int sdm_set_attributes(sdm_t *h, const double *attr_dev, int64_t ld)
{
    SDM_ENTER(h);
    if (!h->valid) return fail(h, SDM_ESTATE, "no valid state loaded");
    if (h->n_attr < 2) return fail(h, SDM_EINVAL, "the handle was created with n_attr = 1");
    int rc = read_ctrl(h);
    if (rc != SDM_OK) return rc;
    const int64_t n = h->ctrl_host->n;
    h->n_ub = n;
    if (n == 0) return SDM_OK;
    if (!attr_dev || ld < n) return fail(h, SDM_EINVAL, "attribute pointer is NULL or ld < n_sd");
    SDM_CUDA(h, cudaMemcpy2DAsync(h->attr, (size_t)h->L.attr_stride * 8, attr_dev, (size_t)ld * 8, (size_t)n * 8,
                                  (size_t)(h->n_attr - 1), cudaMemcpyDeviceToDevice, h->stream));
    SDM_LAUNCH(h, k_check_attr, grid_for(h, n, 256, 8), 256, 0, attr_view(h), (int)n, h->ctrl);
    rc = read_ctrl(h);
    if (rc != SDM_OK) return rc;
    if (h->ctrl_host->invalid) {
        h->valid = false;
        return fail(h, SDM_EINVAL, "attribute validation failed: every value must be finite");
    }
    return SDM_OK;
}

int sdm_get_attributes(sdm_t *h, double *attr_dev, int64_t ld)
{
    SDM_ENTER(h);
    if (!h->valid) return fail(h, SDM_ESTATE, "no valid state loaded");
    if (h->n_attr < 2) return fail(h, SDM_EINVAL, "the handle was created with n_attr = 1");
    int rc = read_ctrl(h);
    if (rc != SDM_OK) return rc;
    const int64_t n = h->ctrl_host->n;
    h->n_ub = n;
    if (n == 0) return SDM_OK;
    if (!attr_dev || ld < n) return fail(h, SDM_EINVAL, "attribute pointer is NULL or ld < n_sd");
    SDM_CUDA(h, cudaMemcpy2DAsync(attr_dev, (size_t)ld * 8, h->attr, (size_t)h->L.attr_stride * 8, (size_t)n * 8,
                                  (size_t)(h->n_attr - 1), cudaMemcpyDeviceToDevice, h->stream));
    SDM_CUDA(h, cudaStreamSynchronize(h->stream));
    return SDM_OK;
}

static int get_state_impl(sdm_t *h, int64_t *n_sd, int64_t *xi, double *v, int32_t *cell, cudaMemcpyKind kind)
{
    SDM_ENTER(h);
    if (!h->valid) return fail(h, SDM_ESTATE, "no valid state loaded");
    int rc = read_ctrl(h);
    if (rc != SDM_OK) return rc;
    int64_t n = h->ctrl_host->n;
    h->n_ub = n;
    if (n_sd) *n_sd = n;
    if (n > 0) {
        if (xi) SDM_CUDA(h, cudaMemcpyAsync(xi, h->xi, (size_t)n * 8, kind, h->stream));
        if (v) SDM_CUDA(h, cudaMemcpyAsync(v, h->v, (size_t)n * 8, kind, h->stream));
        if (cell) SDM_CUDA(h, cudaMemcpyAsync(cell, h->cell, (size_t)n * 4, kind, h->stream));
        SDM_CUDA(h, cudaStreamSynchronize(h->stream));
    }
    return SDM_OK;
}

int sdm_get_state(sdm_t *h, int64_t *n_sd, int64_t *xi_dev, double *v_dev, int32_t *cell_id_dev)
{
    return get_state_impl(h, n_sd, xi_dev, v_dev, cell_id_dev, cudaMemcpyDeviceToDevice);
}

int sdm_get_state_host(sdm_t *h, int64_t *n_sd, int64_t *xi_host, double *v_host, int32_t *cell_id_host)
{
    return get_state_impl(h, n_sd, xi_host, v_host, cell_id_host, cudaMemcpyDeviceToHost);
}

int sdm_coalescence_step(sdm_t *h, double dt, double dV, const sdm_kernel_t *kernel, uint64_t seed, uint64_t step)
{
    SDM_ENTER(h);
    if (!h->valid) return fail(h, SDM_ESTATE, "no valid state loaded");
    StepParams prm;
    int rc = make_params(h, dt, dV, kernel, seed, step, prm);
    if (rc != SDM_OK) return rc;
    rc = enqueue_step(h, prm);
    if (rc == SDM_OK) h->stepped = true;
    return rc;
}

int sdm_coalescence_step_moments(sdm_t *h, double dt, double dV, const sdm_kernel_t *kernel, uint64_t seed,
                                 uint64_t step, int64_t *m0_dev, double *m1_dev, double *m2_dev)
{
    SDM_ENTER(h);
    if (!h->valid) return fail(h, SDM_ESTATE, "no valid state loaded");
    if (!m0_dev || !m1_dev || !m2_dev) return fail(h, SDM_EINVAL, "moment output pointer is NULL");
    StepParams prm;
    int rc = make_params(h, dt, dV, kernel, seed, step, prm);
    if (rc != SDM_OK) return rc;
    rc = enqueue_step(h, prm, m0_dev, m1_dev, m2_dev);
    if (rc == SDM_OK) h->stepped = true;
    return rc;
}

int sdm_remove_zero(sdm_t *h, int64_t *n_sd_out)
{
    SDM_ENTER(h);
    if (!h->valid) return fail(h, SDM_ESTATE, "no valid state loaded");
    int rc = enqueue_remove_zero(h);
    if (rc != SDM_OK) return rc;
    if (n_sd_out) {
        rc = read_ctrl(h);
        if (rc != SDM_OK) return rc;
        h->n_ub = h->ctrl_host->n;
        *n_sd_out = h->n_ub;
    }
    return SDM_OK;
}

int sdm_moments(sdm_t *h, int per_cell, int64_t *m0_dev, double *m1_dev, double *m2_dev)
{
    SDM_ENTER(h);
    if (!h->valid) return fail(h, SDM_ESTATE, "no valid state loaded");
    if (!m0_dev || !m1_dev || !m2_dev) return fail(h, SDM_EINVAL, "moment output pointer is NULL");
    return enqueue_moments(h, per_cell, m0_dev, m1_dev, m2_dev);
}

int sdm_moments_host(sdm_t *h, int per_cell, int64_t *m0_host, double *m1_host, double *m2_host)
{
    SDM_ENTER(h);
    if (!h->valid) return fail(h, SDM_ESTATE, "no valid state loaded");
    if (!m0_host || !m1_host || !m2_host) return fail(h, SDM_EINVAL, "moment output pointer is NULL");
    if (!per_cell) {
        int rc = enqueue_moments(h, 0, h->mom0, h->mom1, h->mom2);
        if (rc != SDM_OK) return rc;
        SDM_CUDA(h, cudaMemcpyAsync(m0_host, h->mom0, 8, cudaMemcpyDeviceToHost, h->stream));
        SDM_CUDA(h, cudaMemcpyAsync(m1_host, h->mom1, 8, cudaMemcpyDeviceToHost, h->stream));
        SDM_CUDA(h, cudaMemcpyAsync(m2_host, h->mom2, 8, cudaMemcpyDeviceToHost, h->stream));
        SDM_CUDA(h, cudaStreamSynchronize(h->stream));
        return SDM_OK;
    }
    // per-cell on the host: stage through idx/order space?  No: keep the ABI simple -- the per-cell
    // host variant needs 20 bytes per cell of device scratch, which we take from `order` and
    // `bucket_start`-independent space only if it fits; otherwise ask for the device variant.
    size_t need = (size_t)h->n_cell * 24;
    if (need > (size_t)h->capacity * 4) return fail(h, SDM_EINVAL, "per-cell host moments need n_cell*24 <= capacity*4 bytes of scratch; use sdm_moments");
    int64_t *d0 = reinterpret_cast<int64_t *>(h->order);
    double *d1 = reinterpret_cast<double *>(h->order) + h->n_cell;
    double *d2 = d1 + h->n_cell;
    int rc = enqueue_moments(h, 1, d0, d1, d2);
    if (rc != SDM_OK) return rc;
    SDM_CUDA(h, cudaMemcpyAsync(m0_host, d0, (size_t)h->n_cell * 8, cudaMemcpyDeviceToHost, h->stream));
    SDM_CUDA(h, cudaMemcpyAsync(m1_host, d1, (size_t)h->n_cell * 8, cudaMemcpyDeviceToHost, h->stream));
    SDM_CUDA(h, cudaMemcpyAsync(m2_host, d2, (size_t)h->n_cell * 8, cudaMemcpyDeviceToHost, h->stream));
    SDM_CUDA(h, cudaStreamSynchronize(h->stream));
    return SDM_OK;
}

int sdm_spectrum(sdm_t *h, int32_t n_bins, const double *v_edges_host, const double *dlnr_host, double rho,
                 double V, int32_t n_smooth, double *out_host)
{
    SDM_ENTER(h);
    if (!h->valid) return fail(h, SDM_ESTATE, "no valid state loaded");
    if (n_bins < 1 || n_bins > SDM_MAX_BINS) return fail(h, SDM_EINVAL, "need 1 <= n_bins <= SDM_MAX_BINS");
    if (!v_edges_host || !dlnr_host || !out_host) return fail(h, SDM_EINVAL, "spectrum pointer is NULL");
    if (!(rho > 0.0) || !(V > 0.0) || !std::isfinite(rho) || !std::isfinite(V) || n_smooth < 0 || n_smooth > 64)
        return fail(h, SDM_EINVAL, "need rho > 0, V > 0, 0 <= n_smooth <= 64");
    for (int b = 0; b <= n_bins; ++b) {
        if (!std::isfinite(v_edges_host[b]) || (b > 0 && !(v_edges_host[b] > v_edges_host[b - 1])))
            return fail(h, SDM_EINVAL, "bin edges must be finite and strictly increasing");
        if (b < n_bins && (!(dlnr_host[b] > 0.0) || !std::isfinite(dlnr_host[b])))
            return fail(h, SDM_EINVAL, "bin widths must be finite and > 0");
    }
    double *edges = h->spec, *dlnr = edges + SDM_MAX_BINS + 1, *sums = dlnr + SDM_MAX_BINS, *out = sums + SDM_MAX_BINS;
    SDM_CUDA(h, cudaMemcpyAsync(edges, v_edges_host, (size_t)(n_bins + 1) * 8, cudaMemcpyHostToDevice, h->stream));
    SDM_CUDA(h, cudaMemcpyAsync(dlnr, dlnr_host, (size_t)n_bins * 8, cudaMemcpyHostToDevice, h->stream));
    SDM_LAUNCH(h, k_spectrum_bin, grid_for(h, h->n_ub, 256, 4), 256, 0, h->xi, h->v, h->ctrl, n_bins, edges, sums);
    SDM_LAUNCH(h, k_spectrum_finish, 1, kMaxBins, 0, n_bins, sums, dlnr, rho, V, n_smooth, out);
    SDM_CUDA(h, cudaMemcpyAsync(out_host, out, (size_t)n_bins * 8, cudaMemcpyDeviceToHost, h->stream));
    SDM_CUDA(h, cudaStreamSynchronize(h->stream));
    return SDM_OK;
}

int sdm_get_permutation(sdm_t *h, int32_t *idx_dev, int32_t *cell_start_dev)
{
    SDM_ENTER(h);
    if (!h->valid) return fail(h, SDM_ESTATE, "no valid state loaded");
    if (!h->stepped) return fail(h, SDM_ESTATE, "no permutation: call sdm_coalescence_step first");
    if (idx_dev) {
        if (!h->write_idx) return fail(h, SDM_ESTATE, "permutation export is switched off (SDM_OPT_WRITE_IDX)");
        int rc = read_ctrl(h);                 // exact n_sd: the caller sized idx_dev by it
        if (rc != SDM_OK) return rc;
        h->n_ub = h->ctrl_host->n;
        if (h->n_ub > 0)
            SDM_CUDA(h, cudaMemcpyAsync(idx_dev, h->idx, (size_t)h->n_ub * 4, cudaMemcpyDeviceToDevice, h->stream));
    }
    if (cell_start_dev)
        SDM_CUDA(h, cudaMemcpyAsync(cell_start_dev, h->cell_start, ((size_t)h->n_cell + 1) * 4,
                                    cudaMemcpyDeviceToDevice, h->stream));
    return SDM_OK;
}

int sdm_run(sdm_t *h, double dt, double dV, const sdm_kernel_t *kernel, uint64_t seed, uint64_t step0,
            int64_t n_steps, int remove_zero_each_step)
{
    SDM_ENTER(h);
    if (!h->valid) return fail(h, SDM_ESTATE, "no valid state loaded");
    if (n_steps < 0) return fail(h, SDM_EINVAL, "n_steps < 0");
    StepParams prm;
    int rc = make_params(h, dt, dV, kernel, seed, step0, prm);
    if (rc != SDM_OK) return rc;
    if (box_ctas(h) > 0 && n_steps > 0) {
        SDM_TIMED(h, { rc = enqueue_box(h, prm, n_steps, remove_zero_each_step ? 1 : 0); if (rc != SDM_OK) return rc; });
        h->stepped = true;
        return SDM_OK;
    }
    for (int64_t s = 0; s < n_steps; ++s) {
        if (remove_zero_each_step) {
            rc = enqueue_remove_zero(h);
            if (rc != SDM_OK) return rc;
        }
        prm.step = step0 + (uint64_t)s;
        rc = enqueue_step(h, prm);
        if (rc != SDM_OK) return rc;
        h->stepped = true;
    }
    return SDM_OK;
}

int sdm_get_timing(sdm_t *h, double *total_ms, int64_t *n_launches)
{
    SDM_ENTER(h);
    if (!total_ms || !n_launches) return SDM_EINVAL;
    SDM_CUDA(h, cudaStreamSynchronize(h->stream));
    double total = 0.0;
    int64_t count = 0;
    for (size_t i = 0; i + 1 < h->ev_used; i += 2) {
        float ms = 0.0f;
        SDM_CUDA(h, cudaEventElapsedTime(&ms, h->ev[i], h->ev[i + 1]));
        total += ms;
        count += 1;
    }
    h->ev_used = 0;
    *total_ms = total;
    *n_launches = count;
    return SDM_OK;
}

int sdm_get_counters(sdm_t *h, int64_t *counters_host)
{
    SDM_ENTER(h);
    if (!counters_host) return SDM_EINVAL;
    int rc = read_ctrl(h);
    if (rc != SDM_OK) return rc;
    for (int i = 0; i < SDM_CNT_COUNT; ++i) counters_host[i] = 0;
    counters_host[SDM_CNT_N_SD] = h->ctrl_host->n;
    counters_host[SDM_CNT_EVENTS] = (int64_t)h->ctrl_host->n_events;
    counters_host[SDM_CNT_ZEROS] = h->ctrl_host->zero_count;
    counters_host[SDM_CNT_LAUNCHES] = h->launches;
    counters_host[SDM_CNT_MODE] = !h->valid ? 0 : (box_ctas(h) > 0 ? 2 : (use_fused(h) ? 1 : 0));
    counters_host[SDM_CNT_MAX_CELL] = h->max_count;
    counters_host[SDM_CNT_EXACT_EVALS] = (int64_t)h->ctrl_host->n_exact;
    if (h->valid) h->n_ub = h->ctrl_host->n;
    return SDM_OK;
}

}  // extern "C"
