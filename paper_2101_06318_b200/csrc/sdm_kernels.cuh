// sdm_kernels.cuh -- CUDA kernels of the SDM coalescence step for sm_100a (rows a1-a8 of the
// hot-path table in DESIGN.md).  Included once by sdm_api.cu.
#pragma once

#include "sdm_device.cuh"

namespace sdmk {

constexpr int kWarpCap = 512;            // largest segment one warp sorts in shared memory
constexpr int kSortWarps = 8;            // warps per CTA in the segment kernels
constexpr int kCompactTile = 2048;       // elements per compaction tile
constexpr int kCompactThreads = 256;
constexpr int kMomentBlocks = 1184;      // grid of k_moments_global: 148 SMs x 8
constexpr int kMomentPartials = 8192;    // per-CTA moment partials (part0..2): the largest grid of ANY kernel that
                                         // ends in moments_finish; every such launch is checked against it on the host
constexpr int kMomentThreads = 256;
constexpr int kCellStartQuads = 4;       // k_cell_start_sorted: 16-byte loads per thread and round

// Device-resident control block: everything the host would otherwise have to synchronise for.
struct Ctrl {
    int n;                         // current number of super-droplets
    int zero_count;                // droplets with xi == 0 in the state
    int ticket;                    // compaction tile ticket
    int n_new;                     // compaction result
    int n_buckets;                 // number of sort segments (split mode)
    int unsorted;                  // analysis: cell_id decreases somewhere
    int invalid;                   // analysis: validation failed
    int max_count;                 // analysis: largest cell
    unsigned int moment_done;      // moments: last-block counter
    unsigned int compact_done;     // compaction: CTAs that have left the kernel
    unsigned int epoch;            // compaction: tag of valid tile status words (no clearing between calls)
    int cell_ticket[2];            // per-cell kernel: dynamic work counters; a launch draws from one and arms the other
                                   // for the launch that follows (no re-arming launch in between)
    int table_dirty;               // fused path: cell_start must be rebuilt from cell_id (compaction moved droplets and
                                   // did not rebuild the table itself)
    unsigned long long n_events;   // pairs with gamma_tilde > 0
    unsigned long long n_exact;    // pairs whose Eq. 3 was evaluated in fp64
    // upper bounds over the WHOLE state for the probability screening of the general and box paths (sdm_general.cuh):
    // xi never grows (Eq. 5-6), so the largest multiplicity at sdm_set_state stays a bound; volumes grow only in
    // coalescence events, which raise v_max_bits (bit pattern of a positive double: ordered like the value)
    long long xi_max;
    unsigned long long v_max_bits;
    int scan_ticket;               // general path scan: tile ticket
    unsigned int scan_done;        // general path scan: CTAs that have left the kernel
    unsigned int scan_epoch;       // general path scan: tag of valid status words
    unsigned int bar_gen;          // k_compact: generation of its grid barrier (compaction -> table rebuild)
};

__device__ __forceinline__ int lane_id() { return threadIdx.x & 31; }

// ---------------------------------------------------------------------------------------------
// sdm_set_state: validation + layout analysis (not on the per-step path)
// ---------------------------------------------------------------------------------------------
__global__ void k_analyze(const int64_t *__restrict__ xi, const double *__restrict__ v,
                          const int32_t *__restrict__ cell, int n, int n_cell,
                          int *__restrict__ cell_cnt, Ctrl *ctrl)
{
    int zeros = 0, bad = 0, unsorted = 0;
    long long xmax = 0;
    unsigned long long vmax = 0ull;
    for (int i0 = (blockIdx.x * blockDim.x + threadIdx.x) & ~31; i0 < n; i0 += gridDim.x * blockDim.x) {
        const int i = i0 + lane_id();
        int c = -1;
        if (i < n) {
            c = cell[i];
            const int64_t x = xi[i];
            const double vol = v[i];
            const bool ok = (c >= 0) && (c < n_cell) && (x >= 0) && (vol > 0.0) && (vol < CUDART_INF);
            if (!ok) { bad = 1; c = -1; }
            else {
                xmax = max(xmax, (long long)x);
                vmax = max(vmax, (unsigned long long)__double_as_longlong(vol));
                zeros += (x == 0);
                if (i > 0 && cell[i - 1] > c) unsorted = 1;
            }
        }
        const unsigned peers = __match_any_sync(0xffffffffu, c);   // one atomic per distinct cell and warp
        if (c >= 0 && (int)(__ffs(peers) - 1) == lane_id()) atomicAdd(&cell_cnt[c], __popc(peers));
    }
    zeros = __reduce_add_sync(0xffffffffu, zeros);
    bad = __any_sync(0xffffffffu, bad);
    unsorted = __any_sync(0xffffffffu, unsorted);
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        xmax = max(xmax, __shfl_xor_sync(0xffffffffu, xmax, d));
        vmax = max(vmax, __shfl_xor_sync(0xffffffffu, vmax, d));
    }
    if (lane_id() == 0) {
        if (zeros) atomicAdd(&ctrl->zero_count, zeros);
        if (bad) atomicOr(&ctrl->invalid, 1);
        if (unsorted) atomicOr(&ctrl->unsorted, 1);
        atomicMax(&ctrl->xi_max, xmax);
        atomicMax(&ctrl->v_max_bits, vmax);
    }
}

// sdm_set_cell_id (NEXT-4): new cell ids for the droplets in storage -- range check, sortedness, counts
__global__ void k_analyze_cells(const int32_t *__restrict__ cell, int n, int n_cell, int *__restrict__ cell_cnt,
                                Ctrl *ctrl)
{
    int bad = 0, unsorted = 0;
    for (int i0 = (blockIdx.x * blockDim.x + threadIdx.x) & ~31; i0 < n; i0 += gridDim.x * blockDim.x) {
        const int i = i0 + lane_id();
        int c = -1;
        if (i < n) {
            c = cell[i];
            if (c < 0 || c >= n_cell) { bad = 1; c = -1; }
            else if (i > 0 && cell[i - 1] > c) unsorted = 1;
        }
        const unsigned peers = __match_any_sync(0xffffffffu, c);
        if (c >= 0 && (int)(__ffs(peers) - 1) == lane_id()) atomicAdd(&cell_cnt[c], __popc(peers));
    }
    bad = __any_sync(0xffffffffu, bad);
    unsorted = __any_sync(0xffffffffu, unsorted);
    if (lane_id() == 0) {
        if (bad) atomicOr(&ctrl->invalid, 1);
        if (unsorted) atomicOr(&ctrl->unsorted, 1);
    }
}

// sdm_set_attributes: every value of the extra attribute rows must be finite
__global__ void k_check_attr(const AttrView av, int n, Ctrl *ctrl)
{
    int bad = 0;
    for (int r = 0; r < av.n; ++r)
        for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
            const double a = av.p[(long long)r * av.stride + i];
            if (!(fabs(a) < CUDART_INF)) bad = 1;
        }
    if (__any_sync(0xffffffffu, bad) && lane_id() == 0) atomicOr(&ctrl->invalid, 1);
}

// also clears the counters (invariant of the general path: cell_cnt[] is zero between kernels that use it)
__global__ void k_max_count(int *__restrict__ cell_cnt, int n_cell, Ctrl *ctrl)
{
    int m = 0;
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < n_cell; c += gridDim.x * blockDim.x) {
        m = max(m, cell_cnt[c]);
        cell_cnt[c] = 0;
    }
    m = __reduce_max_sync(0xffffffffu, m);
    if (lane_id() == 0 && m > 0) atomicMax(&ctrl->max_count, m);
}

// ---------------------------------------------------------------------------------------------
// Row a2 (general path): counting sort by cell -- histogram, scan, scatter
// ---------------------------------------------------------------------------------------------
constexpr int kCellCountBins = 2048;     // up to this many cells the histogram is privatised per CTA

__global__ void __launch_bounds__(256)
k_cell_count(const int32_t *__restrict__ cell, const Ctrl *__restrict__ ctrl, int n_cell,
             int *__restrict__ cell_cnt)
{
    __shared__ int s_cnt[kCellCountBins];
    const int n = ctrl->n;
    const bool priv = n_cell <= kCellCountBins;       // few cells (a box is ONE cell): same-address atomics
    if (priv) {                                       // would serialise in L2, so count in shared memory first
        for (int c = threadIdx.x; c < n_cell; c += blockDim.x) s_cnt[c] = 0;
        __syncthreads();
    }
    // lanes of a warp that hit the same cell (all of them in a single-cell box) send ONE atomic
    for (int i0 = (blockIdx.x * blockDim.x + threadIdx.x) & ~31; i0 < n; i0 += gridDim.x * blockDim.x) {
        const int i = i0 + lane_id();
        const int c = (i < n) ? cell[i] : -1;
        const unsigned peers = __match_any_sync(0xffffffffu, c);
        if (c >= 0 && (int)(__ffs(peers) - 1) == lane_id()) atomicAdd(priv ? &s_cnt[c] : &cell_cnt[c], __popc(peers));
    }
    if (priv) {
        __syncthreads();
        for (int c = threadIdx.x; c < n_cell; c += blockDim.x)
            if (s_cnt[c]) atomicAdd(&cell_cnt[c], s_cnt[c]);
    }
}

// Single-CTA exclusive scan of per-cell counts -> cell_start[n_cell+1].  With split != 0 it also
// decides, per cell, how many key bits sub-divide the cell into sort segments ("buckets": cells
// larger than seg_cap are cut by the top bits of the uniform sort key into pieces of mean size
// in (seg_cap/4, seg_cap/2]) and scans the bucket counts -> bucket_base[n_cell+1].
constexpr int kScanThreads = 1024;
constexpr int kScanItems = 8;

__device__ __forceinline__ int block_exclusive_scan(int val, int *s_warp, int &total)
{
    const int lane = lane_id(), warp = threadIdx.x >> 5;
    int inc = val;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += t;
    }
    __syncthreads();
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        int w = s_warp[lane];
        int winc = w;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, winc, d);
            if (lane >= d) winc += t;
        }
        s_warp[lane] = winc - w;      // exclusive warp offsets
        if (lane == 31) s_warp[32] = winc;
    }
    __syncthreads();
    total = s_warp[32];
    return s_warp[warp] + inc - val;
}

__device__ __forceinline__ int split_bits(int count, int seg_cap)
{
    if (count <= seg_cap) return 0;
    // smallest B with count / 2^B <= seg_cap/2
    int target = max(seg_cap >> 1, 1);
    int B = 0;
    while (((long long)target << B) < count) ++B;
    return B;
}

__global__ void __launch_bounds__(kScanThreads)
k_cell_scan(int *__restrict__ cnt, int n_cell, int *__restrict__ cell_start, int split,
            int seg_cap, int *__restrict__ cell_bits, int *__restrict__ bucket_base, Ctrl *ctrl)
{
    __shared__ int s_warp[33];
    int carry = 0, bcarry = 0;
    for (int base = 0; base < n_cell; base += kScanThreads * kScanItems) {
        int c0 = base + threadIdx.x * kScanItems;
        int loc[kScanItems], nb[kScanItems];
        int sum = 0, bsum = 0;
#pragma unroll
        for (int k = 0; k < kScanItems; ++k) {
            int c = c0 + k;
            loc[k] = (c < n_cell) ? cnt[c] : 0;
            int B = split ? split_bits(loc[k], seg_cap) : 0;
            nb[k] = (c < n_cell) ? (1 << B) : 0;
            if (c < n_cell) cell_bits[c] = B;
            sum += loc[k];
            bsum += nb[k];
        }
        int total, btotal = 0;
        int excl = block_exclusive_scan(sum, s_warp, total);
        int bexcl = block_exclusive_scan(bsum, s_warp, btotal);
        int run = carry + excl, brun = bcarry + bexcl;
#pragma unroll
        for (int k = 0; k < kScanItems; ++k) {
            int c = c0 + k;
            if (c < n_cell) {
                cell_start[c] = run;
                cnt[c] = 0;
                bucket_base[c] = brun;
            }
            run += loc[k];
            brun += nb[k];
        }
        carry += total;
        bcarry += btotal;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        cell_start[n_cell] = carry;
        bucket_base[n_cell] = bcarry;
        ctrl->n_buckets = bcarry;
    }
}

// ---------------------------------------------------------------------------------------------
// Row a3 helpers: exact (key64, storage index) order -- bitonic network in shared memory, ranking by counting
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ bool key_less(uint64_t ka, int ia, uint64_t kb, int ib)
{
    return (ka < kb) || (ka == kb && ia < ib);          // R7: ties by storage index
}

// bitonic sort of (skey[e], sid[e]), e in [0, N), N a power of two, by one warp
__device__ __forceinline__ void warp_bitonic(uint64_t *skey, int *sid, int N, int lane)
{
    for (int k = 2; k <= N; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int t = lane; t < (N >> 1); t += 32) {
                int i = ((t & ~(j - 1)) << 1) | (t & (j - 1));
                int l = i | j;
                bool up = (i & k) == 0;
                uint64_t ka = skey[i], kb = skey[l];
                int ia = sid[i], ib = sid[l];
                bool swap = up ? key_less(kb, ib, ka, ia) : key_less(ka, ia, kb, ib);
                if (swap) { skey[i] = kb; skey[l] = ka; sid[i] = ib; sid[l] = ia; }
            }
            __syncwarp();
        }
    }
}

// Never taken with Philox keys and the default cap (a segment would have to exceed its mean by
// more than 16 standard deviations); kept so that the result is defined for every input:
// rank by counting, O(m^2) Philox evaluations.
__device__ __noinline__ void warp_rank_by_counting(const int *__restrict__ ids_in, int contiguous_base,
                                                   int m, int out_base, int *__restrict__ idx,
                                                   uint64_t step, const PhiloxKey &rk, int lane)
{
    for (int e = lane; e < m; e += 32) {
        int id = ids_in ? ids_in[e] : contiguous_base + e;
        uint64_t key = block_key64(droplet_block_any((uint32_t)id, step, rk));
        int rank = 0;
        for (int f = 0; f < m; ++f) {
            int id2 = ids_in ? ids_in[f] : contiguous_base + f;
            uint64_t key2 = block_key64(droplet_block_any((uint32_t)id2, step, rk));
            rank += key_less(key2, id2, key, id) ? 1 : 0;
        }
        idx[out_base + rank] = id;
    }
}

// ---------------------------------------------------------------------------------------------
// Fused path (cell-contiguous storage): row a2 by boundary detection, rows a1,a3-a6 per cell
// ---------------------------------------------------------------------------------------------
// cell_id is non-decreasing: cell c starts where the id first reaches c.  Every thread inspects four
// consecutive droplets (one 16-byte load) and the one before them; writes happen only at boundaries.
__device__ __forceinline__ void cell_boundary(int prev, int c, int i, int *__restrict__ cell_start)
{
    for (int cc = prev + 1; cc <= c; ++cc) cell_start[cc] = i;     // also fills empty cells
}

// Grid-wide: every thread of every CTA calls it (CTAs of 256 threads).
// kReadOnly = true: `cell` is not written by the launch that calls this (k_cell_start_sorted): streaming loads and the
// non-coherent path (ld.global.nc) for the neighbour look-ups.  kReadOnly = false: the same launch rewrote `cell` in
// place before a grid barrier (k_compact): ld.global.nc is only defined for data that stays read-only for the whole
// kernel, and this SM may hold pre-barrier lines of the same addresses, so every read of `cell` goes to L2 (ld.cg).
template <bool kReadOnly>
__device__ __forceinline__ int4 cell_quad_load(const int4 *p) { return kReadOnly ? __ldcs(p) : __ldcg(p); }
template <bool kReadOnly>
__device__ __forceinline__ int cell_id_load(const int32_t *p) { return kReadOnly ? __ldg(p) : __ldcg(p); }

template <bool kReadOnly>
__device__ __forceinline__ void cell_start_rebuild(const int32_t *cell, const Ctrl *ctrl, int n_cell,
                                                   int *__restrict__ cell_start)
{
    const int n = ((volatile const Ctrl *)ctrl)->n;
    if (n == 0) {
        for (int c = blockIdx.x * blockDim.x + threadIdx.x; c <= n_cell; c += gridDim.x * blockDim.x)
            cell_start[c] = 0;
        return;
    }
    const int n4 = (n + 3) >> 2;
    const int4 *cell4 = reinterpret_cast<const int4 *>(cell);
    const int T = blockDim.x, lane = lane_id();                     // a CTA reads U*T consecutive quads per round
    constexpr int U = kCellStartQuads;                              // independent 16-byte loads in flight per thread
    for (int t0 = blockIdx.x * (U * T) + threadIdx.x; t0 - lane < n4; t0 += gridDim.x * (U * T)) {
        const int t_hi = t0 - lane + 31 + (U - 1) * T;              // the largest quad index this warp touches
        if (t_hi < n4 - 1 && t0 - lane > 0) {
            // fast path (warp-uniform): every quad is complete and none is the first or the last
            int4 q[U];
            int pv[U];
#pragma unroll
            for (int u = 0; u < U; ++u) q[u] = cell_quad_load<kReadOnly>(cell4 + t0 + u * T);
#pragma unroll
            for (int u = 0; u < U; ++u) pv[u] = (lane == 0) ? cell_id_load<kReadOnly>(cell + ((t0 + u * T) << 2) - 1) : 0;
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int i = (t0 + u * T) << 2;
                int prev = __shfl_up_sync(0xffffffffu, q[u].w, 1);  // the droplet before this thread's four
                if (lane == 0) prev = pv[u];
                if (prev != q[u].w) {                               // some boundary among the four
                    if (q[u].x != prev) cell_boundary(prev, q[u].x, i, cell_start);
                    if (q[u].y != q[u].x) cell_boundary(q[u].x, q[u].y, i + 1, cell_start);
                    if (q[u].z != q[u].y) cell_boundary(q[u].y, q[u].z, i + 2, cell_start);
                    if (q[u].w != q[u].z) cell_boundary(q[u].z, q[u].w, i + 3, cell_start);
                }
            }
            continue;
        }
        for (int u = 0; u < U; ++u) {                               // edges of the array
            const int t = t0 + u * T, i = t << 2;
            if (t >= n4) break;
            int c0, c1, c2, c3;
            if (i + 3 < n) {
                const int4 q = cell_quad_load<kReadOnly>(cell4 + t);
                c0 = q.x; c1 = q.y; c2 = q.z; c3 = q.w;
            } else {                                                // the last, partial quad: repeat the last id
                c0 = cell_id_load<kReadOnly>(cell + i);
                c1 = (i + 1 < n) ? cell_id_load<kReadOnly>(cell + i + 1) : c0;
                c2 = (i + 2 < n) ? cell_id_load<kReadOnly>(cell + i + 2) : c1;
                c3 = c2;
            }
            const int prev = (i > 0) ? cell_id_load<kReadOnly>(cell + i - 1) : -1;
            if (prev != c3) {
                if (c0 != prev) cell_boundary(prev, c0, i, cell_start);
                if (c1 != c0) cell_boundary(c0, c1, i + 1, cell_start);
                if (c2 != c1) cell_boundary(c1, c2, i + 2, cell_start);
                if (c3 != c2) cell_boundary(c2, c3, i + 3, cell_start);
            }
            if (i + 4 >= n)                                         // the thread holding the last droplet
                for (int cc = c3 + 1; cc <= n_cell; ++cc) cell_start[cc] = n;
        }
    }
}

// Builds the table the fused path's first step after sdm_set_state / sdm_set_cell_id reads (later tables come out of
// the step kernel itself, and out of k_compact when a compaction moves droplets); arms the chunk ticket of that step.
__global__ void __launch_bounds__(256)
k_cell_start_sorted(const int32_t *__restrict__ cell, Ctrl *ctrl, int n_cell, int *__restrict__ cell_start, int ticket_sel,
                    int ticket0)
{
    if (blockIdx.x == 0 && threadIdx.x == 0) { ctrl->cell_ticket[ticket_sel] = ticket0; ctrl->table_dirty = 0; }
    cell_start_rebuild<true>(cell, ctrl, n_cell, cell_start);
}

// arms a chunk ticket when the step kernel's grid differs from the one the previous launch armed it for
__global__ void k_arm_ticket(Ctrl *ctrl, int ticket_sel, int ticket0)
{
    ctrl->cell_ticket[ticket_sel] = ticket0;
}

// ---------------------------------------------------------------------------------------------
// Row a7: stable in-place stream compaction of xi == 0 (single pass, decoupled look-back)
// ---------------------------------------------------------------------------------------------
// A tile's aggregate is published only after the whole tile sits in shared memory, and a tile
// learns its output offset only after every earlier tile has published: so by the time a tile
// writes into the (earlier) storage positions, everything there has been read.  Tiles are handed
// out in order by a ticket, which guarantees forward progress of the look-back.
// A tile status word is  epoch (30 bits) | flag (2 bits) | count (32 bits); words of earlier calls carry
// an older epoch and read as "not published", so the array never has to be cleared.
constexpr unsigned long long kFlagAggregate = 1ull << 32, kFlagInclusive = 2ull << 32;

// The pass itself, as a device function, so that the persistent box kernel (sdm_box.cuh) can run it between two steps
// of one launch: called by kCompactThreads threads of every CTA of the grid (tid = their index, n_ctas = the grid size);
// `sync` synchronises exactly those threads (__syncthreads() in k_compact, a named barrier in the box kernel).
struct CompactSmem {
    int64_t s_xi[kCompactTile];
    double s_v[kCompactTile];
    int32_t s_c[kCompactTile];
    int s_warp_cnt[kCompactThreads / 32];
    int s_tile, s_prefix;
};

// grid_wait (k_compact with a table to rebuild; needs every CTA of the launch resident): nobody returns before the last CTA
// has published the new count -- a grid barrier, released through Ctrl::bar_gen.  table_rebuilt: the caller rebuilds the
// fused path's cell table right after, so the table is not left marked dirty.
template <class Sync>
__device__ __forceinline__ void compact_tiles(int64_t *__restrict__ xi, double *__restrict__ v, int32_t *__restrict__ cell,
                                              Ctrl *ctrl, unsigned long long *__restrict__ status, const AttrView &av,
                                              CompactSmem &sm, double *s_extra, int tid, unsigned int n_ctas, Sync sync,
                                              bool grid_wait = false)
{
    const int n = ((volatile Ctrl *)ctrl)->n;
    const unsigned long long tag = (unsigned long long)(((volatile Ctrl *)ctrl)->epoch & 0x3fffffffu) << 34;
    const int n_tiles = (n + kCompactTile - 1) / kCompactTile;
    const int lane = tid & 31, warp = tid >> 5;
    constexpr int kItems = kCompactTile / kCompactThreads;      // 8
    constexpr int kWarpSpan = 32 * kItems;                       // 256 consecutive elements per warp
    while (true) {
        sync();
        if (tid == 0) sm.s_tile = atomicAdd(&ctrl->ticket, 1);
        sync();
        const int tile = sm.s_tile;
        if (tile >= n_tiles) break;
        const int base = tile * kCompactTile;
        const int cnt = min(kCompactTile, n - base);
#pragma unroll
        for (int k = 0; k < kItems; ++k) {
            int e = k * kCompactThreads + tid;
            if (e < cnt) { sm.s_xi[e] = xi[base + e]; sm.s_v[e] = v[base + e]; sm.s_c[e] = cell[base + e]; }
        }
        for (int r = 0; r < av.n; ++r) {                // staged BEFORE the tile publishes its count, like xi and v
            const double *A = av.p + (long long)r * av.stride + base;
#pragma unroll
            for (int k = 0; k < kItems; ++k) {
                int e = k * kCompactThreads + tid;
                if (e < cnt) s_extra[r * kCompactTile + e] = A[e];
            }
        }
        sync();
        unsigned masks[kItems];
        int wtotal = 0;
#pragma unroll
        for (int k = 0; k < kItems; ++k) {
            int e = warp * kWarpSpan + k * 32 + lane;
            bool keep = (e < cnt) && (sm.s_xi[e] != 0);
            masks[k] = __ballot_sync(0xffffffffu, keep);
            wtotal += __popc(masks[k]);
        }
        if (lane == 0) sm.s_warp_cnt[warp] = wtotal;
        sync();
        int woff = 0, tile_total = 0;
#pragma unroll
        for (int w = 0; w < kCompactThreads / 32; ++w) {
            int cw = sm.s_warp_cnt[w];
            if (w < warp) woff += cw;
            tile_total += cw;
        }
        if (tid == 0) {
            int excl = 0;
            volatile unsigned long long *vs = status;
            __threadfence();
            if (tile == 0) {
                vs[0] = tag | kFlagInclusive | (unsigned long long)tile_total;
            } else {
                vs[tile] = tag | kFlagAggregate | (unsigned long long)tile_total;
                int t = tile - 1;
                while (true) {
                    const unsigned long long st = vs[t];
                    if ((st >> 34) != (tag >> 34) || ((st >> 32) & 3ull) == 0) continue;   // not published yet
                    excl += (int)(st & 0xffffffffull);
                    if (((st >> 32) & 3ull) == 2) break;
                    --t;
                }
                vs[tile] = tag | kFlagInclusive | (unsigned long long)(excl + tile_total);
            }
            __threadfence();
            sm.s_prefix = excl;
            if (tile == n_tiles - 1) ctrl->n_new = excl + tile_total;
        }
        sync();
        const int prefix = sm.s_prefix;
        int run = woff;
#pragma unroll
        for (int k = 0; k < kItems; ++k) {
            int e = warp * kWarpSpan + k * 32 + lane;
            if ((masks[k] >> lane) & 1u) {
                int dst = prefix + run + __popc(masks[k] & ((1u << lane) - 1u));
                xi[dst] = sm.s_xi[e];
                v[dst] = sm.s_v[e];
                cell[dst] = sm.s_c[e];
                for (int r = 0; r < av.n; ++r) av.p[(long long)r * av.stride + dst] = s_extra[r * kCompactTile + e];
            }
            run += __popc(masks[k]);
        }
    }
    // the last CTA to leave publishes the new count and re-arms the control block; every CTA has read
    // zero_count and n before it counts itself out, so nobody sees the new values half-way
    sync();
    if (tid == 0) {
        const unsigned int gen = ((volatile Ctrl *)ctrl)->bar_gen;      // read before this CTA counts itself out
        __threadfence();
        if (atomicAdd(&ctrl->compact_done, 1u) == n_ctas - 1) {
            __threadfence();
            ctrl->n = (n_tiles > 0) ? ((volatile Ctrl *)ctrl)->n_new : 0;
            ctrl->table_dirty = grid_wait ? 0 : 1;
            ctrl->zero_count = 0;
            ctrl->ticket = 0;
            ctrl->compact_done = 0;
            ctrl->epoch = ctrl->epoch + 1u;
            __threadfence();
            ((volatile Ctrl *)ctrl)->bar_gen = gen + 1u;
        } else if (grid_wait) {
            while (((volatile Ctrl *)ctrl)->bar_gen == gen) __nanosleep(64);
        }
        __threadfence();
    }
    if (grid_wait) sync();
}

__global__ void __launch_bounds__(kCompactThreads)
k_compact(int64_t *__restrict__ xi, double *__restrict__ v, int32_t *__restrict__ cell, Ctrl *ctrl,
          unsigned long long *__restrict__ status, const AttrView av, int *__restrict__ next_table, int n_cell)
{
    extern __shared__ double s_extra[];                // av.n rows of kCompactTile values (extra attributes)
    __shared__ CompactSmem sm;
    // nothing to remove: every CTA leaves (zero_count is cleared only after every CTA of a launch has read it)
    if (((volatile Ctrl *)ctrl)->zero_count == 0) return;
    // next_table (fused path, the host launches no more than the resident number of CTAs): the table the next step
    // reads is rebuilt from the compacted cell ids in this launch, behind a grid barrier
    compact_tiles(xi, v, cell, ctrl, status, av, sm, s_extra, (int)threadIdx.x, gridDim.x, [] { __syncthreads(); },
                  next_table != nullptr);
    if (next_table != nullptr) cell_start_rebuild<false>(cell, ctrl, n_cell, next_table);   // `cell` was rewritten above
}

// ---------------------------------------------------------------------------------------------
// Row a8: moments M0 = sum xi (int64), M1 = sum xi v, M2 = sum xi v^2 (fp64)
// ---------------------------------------------------------------------------------------------
// CTA-level finish shared by the moment kernels: per-thread partial sums -> one partial per CTA ->
// the last CTA to arrive sums all partials in a fixed order (run-to-run deterministic) and writes
// the three results.  Every thread of the CTA must call it.
__device__ __forceinline__ void moments_finish(int64_t a0, double a1, double a2, Ctrl *ctrl,
                                               int64_t *__restrict__ part0, double *__restrict__ part1,
                                               double *__restrict__ part2, int64_t *__restrict__ m0,
                                               double *__restrict__ m1, double *__restrict__ m2)
{
    constexpr int kMaxWarps = 32;
    __shared__ int64_t s0[kMaxWarps];
    __shared__ double s1[kMaxWarps], s2[kMaxWarps];
    __shared__ bool s_last;
    const int lane = lane_id(), warp = threadIdx.x >> 5, n_warps = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        a0 += __shfl_down_sync(0xffffffffu, a0, d);
        a1 += __shfl_down_sync(0xffffffffu, a1, d);
        a2 += __shfl_down_sync(0xffffffffu, a2, d);
    }
    if (lane == 0) { s0[warp] = a0; s1[warp] = a1; s2[warp] = a2; }
    __syncthreads();
    if (threadIdx.x == 0) {
        int64_t b0 = 0;
        double b1 = 0.0, b2 = 0.0;
        for (int w = 0; w < n_warps; ++w) { b0 += s0[w]; b1 += s1[w]; b2 += s2[w]; }
        part0[blockIdx.x] = b0; part1[blockIdx.x] = b1; part2[blockIdx.x] = b2;
        __threadfence();
        unsigned int done = atomicAdd(&ctrl->moment_done, 1u);
        s_last = (done == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    a0 = 0; a1 = 0.0; a2 = 0.0;
    for (int b = threadIdx.x; b < (int)gridDim.x; b += blockDim.x) {
        a0 += ((volatile int64_t *)part0)[b];
        a1 += ((volatile double *)part1)[b];
        a2 += ((volatile double *)part2)[b];
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        a0 += __shfl_down_sync(0xffffffffu, a0, d);
        a1 += __shfl_down_sync(0xffffffffu, a1, d);
        a2 += __shfl_down_sync(0xffffffffu, a2, d);
    }
    __syncthreads();
    if (lane == 0) { s0[warp] = a0; s1[warp] = a1; s2[warp] = a2; }
    __syncthreads();
    if (threadIdx.x == 0) {
        int64_t b0 = 0;
        double b1 = 0.0, b2 = 0.0;
        for (int w = 0; w < n_warps; ++w) { b0 += s0[w]; b1 += s1[w]; b2 += s2[w]; }
        *m0 = b0; *m1 = b1; *m2 = b2;
        ctrl->moment_done = 0;
    }
}

__global__ void __launch_bounds__(kMomentThreads)
k_moments_global(const int64_t *__restrict__ xi, const double *__restrict__ v, Ctrl *ctrl,
                 int64_t *__restrict__ part0, double *__restrict__ part1, double *__restrict__ part2,
                 int64_t *__restrict__ m0, double *__restrict__ m1, double *__restrict__ m2)
{
    const int n = ctrl->n;
    int64_t a0 = 0;
    double a1 = 0.0, a2 = 0.0;
    // two droplets per thread and iteration: 16-byte loads (both arrays are 256-byte aligned)
    const int n2 = n >> 1;
    const longlong2 *xi2 = reinterpret_cast<const longlong2 *>(xi);
    const double2 *v2 = reinterpret_cast<const double2 *>(v);
    for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < n2; t += gridDim.x * blockDim.x) {
        const longlong2 x = __ldcs(xi2 + t);
        const double2 vol = __ldcs(v2 + t);
        const double xv0 = __dmul_rn(__ll2double_rn(x.x), vol.x), xv1 = __dmul_rn(__ll2double_rn(x.y), vol.y);
        a0 += x.x + x.y;
        a1 = __dadd_rn(a1, __dadd_rn(xv0, xv1));
        a2 = __dadd_rn(a2, __dadd_rn(__dmul_rn(xv0, vol.x), __dmul_rn(xv1, vol.y)));
    }
    if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
        const int64_t x = xi[n - 1];
        const double vol = v[n - 1];
        const double xv = __dmul_rn(__ll2double_rn(x), vol);
        a0 += x;
        a1 = __dadd_rn(a1, xv);
        a2 = __dadd_rn(a2, __dmul_rn(xv, vol));
    }
    moments_finish(a0, a1, a2, ctrl, part0, part1, part2, m0, m1, m2);
}

__global__ void k_moments_zero(int n_cell, int64_t *__restrict__ m0, double *__restrict__ m1,
                               double *__restrict__ m2)
{
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < n_cell; c += gridDim.x * blockDim.x) {
        m0[c] = 0; m1[c] = 0.0; m2[c] = 0.0;
    }
}

// any storage order: atomics per cell (the fp64 sums are then order-dependent in the last bits)
__global__ void k_moments_cell_atomic(const int64_t *__restrict__ xi, const double *__restrict__ v,
                                      const int32_t *__restrict__ cell, const Ctrl *__restrict__ ctrl,
                                      int64_t *__restrict__ m0, double *__restrict__ m1,
                                      double *__restrict__ m2)
{
    const int n = ctrl->n;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        int64_t x = xi[i];
        double vol = v[i];
        int c = cell[i];
        double xv = __dmul_rn(__ll2double_rn(x), vol);
        atomicAdd(reinterpret_cast<unsigned long long *>(&m0[c]), (unsigned long long)x);
        atomicAdd(&m1[c], xv);
        atomicAdd(&m2[c], __dmul_rn(xv, vol));
    }
}

}  // namespace sdmk
