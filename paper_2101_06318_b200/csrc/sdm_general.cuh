// sdm_general.cuh -- general path (any storage order, cells of any size): counting sort by cell / key
// bucket, per-segment sort, pairs.
//
// A "segment" is a cell, or -- for cells larger than the warp capacity -- the droplets of a cell whose
// sort key has the same top B bits (split_bits in sdm_kernels.cuh; k_gen_count, k_gen_scatter below).  order[]
// lists the storage indices of every segment contiguously; this kernel puts each segment into
// (key64, storage index) order (row a3; R6-R7) and writes idx.
//
// One warp per segment of up to 256 droplets, the same O(n) scheme as sdm_fused_count.cuh: counting sort
// on the leading byte of the key, then odd-even transposition rounds in registers.  Inside a segment
// of a split cell the top B key bits are equal, so the sort word is taken from the key shifted left by
// B bits.  Differences from the cell-contiguous kernel: storage indices are gathered through order[]
// (Philox counters and the index written to idx are the gathered ids), and a segment whose truncated
// sort words tie is redone exactly by a bitonic network on the full (key64, index) pairs in shared
// memory.  Segments above 256 droplets (only with SDM_OPT_SEGMENT_CAP, or an astronomically unlikely
// bucket) are ranked by counting.
#pragma once

#include "sdm_fused_count.cuh"

namespace sdmk {

constexpr int kGenWarps = 8;
constexpr int kRankStride = 8;             // rank counters sit one per 32-byte sector: L2 serialises the returning
                                          // atomics that hit one sector (measured: k_gen_count 23 -> 8 us at 2^20)
constexpr int kGenCap = 256;              // segment capacity of the warp counting sort

struct __align__(1024) GenSmem {
    uint32_t cnt[256];                    // histogram in byte units (zero between segments)
    uint32_t start[256];                  // shared-space byte address of each bin's first slot
    uint32_t slot[kGenCap];               // words grouped by bin
    int ids[kGenCap];                     // storage index of local droplet e
    int sid[kGenCap];                     // sorted storage indices (input of the pair loop)
    // exact path (truncated words tie): the full 64-bit keys reuse start[] and slot[], which are dead by then
    __device__ uint64_t *key() { return reinterpret_cast<uint64_t *>(start); }
};
static_assert(sizeof(GenSmem) % 1024 == 0, "GenSmem must tile shared memory in 1 KB units");
static_assert(offsetof(GenSmem, start) == 1024 && offsetof(GenSmem, slot) == 2048, "layout used by the address arithmetic");

constexpr size_t kGenSmemBytes = kGenWarps * sizeof(GenSmem);

// Sort words of one segment: x[k] belongs to local droplet k*32+lane on entry (id[k] its storage index),
// and to sorted position 8*lane+k on return.  shift = key bits shared by the whole segment.
// E = 8 (segments up to 256) or 4 (up to 128: half the Philox blocks and sort words per warp).
template <int E>
__device__ __forceinline__ void count_sort_ids(const int (&id)[E], int m, int lane, int shift, uint64_t step,
                                               const PhiloxKey &rk, GenSmem *sm, uint32_t sm_base, uint32_t (&x)[E])
{
    constexpr int L = 32, N = L * E;
    static_assert(E == 4 || E == 8, "rows per lane");
    const int nrem = m - lane;
    uint32_t old[E];
#pragma unroll
    for (int k = 0; k < E; ++k) {
        x[k] = 0xFFFFFFFFu;
        old[k] = 0;
        if (L * k < m) {                                               // warp-uniform: rows beyond the segment cost nothing
            const bool valid = nrem > L * k;
            const uint4 w = droplet_block_any((uint32_t)id[k], step, rk);
            const uint32_t hi = __funnelshift_l(w.x, w.y, shift);      // top 32 bits of key64 << shift
            if (valid) {
                x[k] = (hi & ~(uint32_t)(N - 1)) | (uint32_t)(lane + L * k);
                old[k] = atoms_add(sm_base | ((hi >> 22) & 0x3FCu), 4u);
            }
        }
    }
    __syncwarp();
    uint32_t rounds;
    {
        uint4 *cnt4 = reinterpret_cast<uint4 *>(sm->cnt);
        const uint4 c0 = cnt4[2 * lane], c1 = cnt4[2 * lane + 1];
        cnt4[2 * lane] = make_uint4(0u, 0u, 0u, 0u);
        cnt4[2 * lane + 1] = make_uint4(0u, 0u, 0u, 0u);
        const uint32_t e1 = c0.x, e2 = e1 + c0.y, e3 = e2 + c0.z, e4 = e3 + c0.w;
        const uint32_t e5 = e4 + c1.x, e6 = e5 + c1.y, e7 = e6 + c1.z, tot = e7 + c1.w;
        const uint32_t cmax = max(max(max(c0.x, c0.y), max(c0.z, c0.w)), max(max(c1.x, c1.y), max(c1.z, c1.w)));
        uint32_t inc = tot;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, inc, d);
            if (lane >= d) inc += t;
        }
        const uint32_t base = (inc - tot) + (sm_base + 2048u);
        uint4 *start4 = reinterpret_cast<uint4 *>(sm->start);
        start4[2 * lane] = make_uint4(base, base + e1, base + e2, base + e3);
        start4[2 * lane + 1] = make_uint4(base + e4, base + e5, base + e6, base + e7);
        rounds = __reduce_max_sync(0xffffffffu, cmax) >> 2;
    }
    __syncwarp();
#pragma unroll
    for (int k = 0; k < E; ++k) {
        if (nrem > L * k) {
            uint32_t dst;
            asm volatile("ld.shared.u32 %0, [%1+1024];" : "=r"(dst) : "r"(sm_base | ((x[k] >> 22) & 0x3FCu)));
            asm volatile("st.shared.u32 [%0], %1;" :: "r"(dst + old[k]), "r"(x[k]) : "memory");
        } else {
            sm->slot[L * k + lane] = 0xFFFFFFFFu;                      // sentinels fill the tail
        }
    }
    __syncwarp();
#pragma unroll
    for (int q = 0; q < E / 4; ++q) {
        const uint4 w = reinterpret_cast<const uint4 *>(sm->slot)[(E / 4) * lane + q];
        x[4 * q] = w.x; x[4 * q + 1] = w.y; x[4 * q + 2] = w.z; x[4 * q + 3] = w.w;
    }
    for (uint32_t r = 0; r < rounds; r += 2) {
#pragma unroll
        for (int k = 0; k + 1 < E; k += 2) cex(x[k], x[k + 1]);
        uint32_t nx0 = __shfl_down_sync(0xffffffffu, x[0], 1);
        uint32_t pxl = __shfl_up_sync(0xffffffffu, x[E - 1], 1);
        if (lane == 31) nx0 = 0xFFFFFFFFu;
        if (lane == 0) pxl = 0u;
#pragma unroll
        for (int k = 1; k + 1 < E; k += 2) cex(x[k], x[k + 1]);
        x[E - 1] = min(x[E - 1], nx0);
        x[0] = max(x[0], pxl);
    }
}

// ---------------------------------------------------------------------------------------------
// Per-step pipeline of the general path:  k_gen_count -> k_gen_scan -> k_gen_scatter ->
// k_segment_sort_pairs (-> k_pairs_straddle when cells are split).
//
// The split of large cells (cell_bits[c] = B key bits, bucket_base[c] = first segment of cell c) is
// decided ONCE per loaded state from the cell counts (k_cell_scan with split = 1): cells never grow
// (PAPER.md:9, 77), so the segments only get smaller afterwards, and idx does not depend on B.
// Invariant between steps: cell_cnt[] and the rank counters are all zero (the scan clears what it read).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ int segment_of(int c, uint32_t key_hi, const int *__restrict__ cell_bits,
                                          const int *__restrict__ bucket_base)
{
    const int B = cell_bits[c];
    return bucket_base[c] + (B > 0 ? (int)(key_hi >> (32 - B)) : 0);
}

// Row a2: per-cell counts and, when cells are split, per-segment counts (needs the droplet's Philox block,
// row a1).  The counting atomic that a droplet's segment receives also RETURNS the droplet's arrival rank in
// that segment (rank[i]), so the scatter pass needs no atomics of its own.  Lanes of a warp that hit the same
// counter send one atomic (a box is ONE cell: same-address atomics would serialise in L2); cell counters that
// are not needed for ranks (split mode) are CTA-privatised in shared memory when there are few cells.
__global__ void __launch_bounds__(256)
k_gen_count(const int32_t *__restrict__ cell, const Ctrl *__restrict__ ctrl, int n_cell, int split,
            const int *__restrict__ cell_bits, const int *__restrict__ bucket_base,
            int *__restrict__ cell_cnt, int *__restrict__ rank_cnt, int *__restrict__ rank,
            const __grid_constant__ StepParams prm)
{
    __shared__ int s_cnt[kCellCountBins];
    const int n = ctrl->n;
    const int lane = lane_id();
    const bool priv = split && n_cell <= kCellCountBins;
    if (priv) {
        for (int c = threadIdx.x; c < n_cell; c += blockDim.x) s_cnt[c] = 0;
        __syncthreads();
    }
    for (int i0 = (blockIdx.x * blockDim.x + threadIdx.x) & ~31; i0 < n; i0 += gridDim.x * blockDim.x) {
        const int i = i0 + lane;
        const int c = (i < n) ? cell[i] : -1;
        const unsigned peers = __match_any_sync(0xffffffffu, c);
        const bool leader = (int)(__ffs(peers) - 1) == lane;
        if (!split) {                                   // segment == cell: the cell counter gives the rank
            int base = 0;
            if (c >= 0 && leader) base = atomicAdd(&rank_cnt[(size_t)c * kRankStride], __popc(peers));
            base = __shfl_sync(0xffffffffu, base, __ffs(peers) - 1);
            if (c >= 0) rank[i] = base + __popc(peers & ((1u << lane) - 1u));
        } else {
            if (c >= 0 && leader) atomicAdd(priv ? &s_cnt[c] : &cell_cnt[c], __popc(peers));
            int seg = -1;
            if (c >= 0) {
                const uint4 w = droplet_block_any((uint32_t)i, prm.step, prm.rk);
                seg = segment_of(c, w.y, cell_bits, bucket_base);
            }
            const unsigned speers = __match_any_sync(0xffffffffu, seg);
            int base = 0;
            if (seg >= 0 && (int)(__ffs(speers) - 1) == lane) base = atomicAdd(&rank_cnt[(size_t)seg * kRankStride], __popc(speers));
            base = __shfl_sync(0xffffffffu, base, __ffs(speers) - 1);
            if (seg >= 0) rank[i] = base + __popc(speers & ((1u << lane) - 1u));
        }
    }
    if (priv) {
        __syncthreads();
        for (int c = threadIdx.x; c < n_cell; c += blockDim.x)
            if (s_cnt[c]) atomicAdd(&cell_cnt[c], s_cnt[c]);
    }
}

// Exclusive scans: cell counts -> cell_start[n_cell+1] and (split) segment counts -> seg_start[n_seg+1].
// Clears the counters it reads.  Tiles of 2048 counters, coalesced loads and stores through shared memory,
// chained by decoupled look-back (tiles handed out in order by a ticket, epoch-tagged status words as in
// k_compact); the two tables are two independent chains of one launch.  A single-CTA scan took 13-22 us for
// 16 K counters (one SM's load/store path); this one is at the launch floor.
constexpr int kScanTile = 2048;
constexpr int kScanTileThreads = 256;

__global__ void __launch_bounds__(kScanTileThreads)
k_gen_scan(int *__restrict__ cell_cnt, int cell_stride, int n_cell, int *__restrict__ cell_start, int split,
           int *__restrict__ seg_cnt, int seg_stride, int n_seg, int *__restrict__ seg_start, Ctrl *ctrl,
           unsigned long long *__restrict__ status)
{
    constexpr int kItems = kScanTile / kScanTileThreads;          // 8
    __shared__ int s_val[kScanTile + kScanTile / 32];             // padded: index e + e/32
    __shared__ int s_warp[kScanTileThreads / 32];
    __shared__ int s_tile, s_prefix;
    const int tid = threadIdx.x, lane = lane_id(), warp = tid >> 5;
    const int tiles_a = (n_cell + kScanTile - 1) / kScanTile;
    const int tiles_b = split ? (n_seg + kScanTile - 1) / kScanTile : 0;
    const unsigned long long tag = (unsigned long long)(ctrl->scan_epoch & 0x3fffffffu) << 34;
    while (true) {
        __syncthreads();
        if (tid == 0) s_tile = atomicAdd(&ctrl->scan_ticket, 1);
        __syncthreads();
        const int tile = s_tile;
        if (tile >= tiles_a + tiles_b) break;
        const bool second = tile >= tiles_a;
        int *cnt = second ? seg_cnt : cell_cnt;
        const size_t stride = second ? seg_stride : cell_stride;
        int *start = second ? seg_start : cell_start;
        const int m = second ? n_seg : n_cell;
        const int chain0 = second ? tiles_a : 0;                  // first tile of this chain
        const int base = (tile - chain0) * kScanTile;
#pragma unroll
        for (int k = 0; k < kItems; ++k) {
            const int e = k * kScanTileThreads + tid;
            s_val[e + (e >> 5)] = (base + e < m) ? cnt[(size_t)(base + e) * stride] : 0;
        }
        __syncthreads();
        int loc[kItems], sum = 0;
#pragma unroll
        for (int k = 0; k < kItems; ++k) {
            const int e = tid * kItems + k;
            loc[k] = s_val[e + (e >> 5)];
            sum += loc[k];
        }
        int inc = sum;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, inc, d);
            if (lane >= d) inc += t;
        }
        if (lane == 31) s_warp[warp] = inc;
        __syncthreads();
        int woff = 0, tile_total = 0;
#pragma unroll
        for (int w = 0; w < kScanTileThreads / 32; ++w) {
            const int cw = s_warp[w];
            if (w < warp) woff += cw;
            tile_total += cw;
        }
        if (tid == 0) {
            int excl = 0;
            volatile unsigned long long *vs = status;
            __threadfence();
            if (tile == chain0) {
                vs[tile] = tag | kFlagInclusive | (unsigned long long)(unsigned int)tile_total;
            } else {
                vs[tile] = tag | kFlagAggregate | (unsigned long long)(unsigned int)tile_total;
                int t = tile - 1;
                while (true) {
                    const unsigned long long st = vs[t];
                    if ((st >> 34) != (tag >> 34) || ((st >> 32) & 3ull) == 0) continue;   // not published yet
                    excl += (int)(st & 0xffffffffull);
                    if (((st >> 32) & 3ull) == 2) break;
                    --t;
                }
                vs[tile] = tag | kFlagInclusive | (unsigned long long)(unsigned int)(excl + tile_total);
            }
            __threadfence();
            s_prefix = excl;
        }
        __syncthreads();
        int run = s_prefix + woff + inc - sum;
#pragma unroll
        for (int k = 0; k < kItems; ++k) {
            const int e = tid * kItems + k;
            s_val[e + (e >> 5)] = run;
            run += loc[k];
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < kItems; ++k) {
            const int e = k * kScanTileThreads + tid;
            if (base + e < m) { start[base + e] = s_val[e + (e >> 5)]; cnt[(size_t)(base + e) * stride] = 0; }
        }
        if (tid == 0 && base + kScanTile >= m) start[m] = s_prefix + tile_total;      // the chain's last tile
    }
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        if (atomicAdd(&ctrl->scan_done, 1u) == gridDim.x - 1) {
            __threadfence();
            ctrl->scan_ticket = 0;
            ctrl->scan_done = 0;
            ctrl->scan_epoch = ctrl->scan_epoch + 1u;
        }
    }
}

// order[] = storage indices grouped by segment, at the arrival rank k_gen_count handed out (any order inside a
// segment would do; the sort makes it unique).
__global__ void __launch_bounds__(256)
k_gen_scatter(const int32_t *__restrict__ cell, const Ctrl *__restrict__ ctrl, int split,
              const int *__restrict__ cell_bits, const int *__restrict__ bucket_base,
              const int *__restrict__ seg_start, const int *__restrict__ rank, int *__restrict__ order,
              const __grid_constant__ StepParams prm)
{
    const int n = ctrl->n;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const int c = cell[i];
        int b = c;
        if (split) {
            const uint4 w = droplet_block_any((uint32_t)i, prm.step, prm.rk);
            b = segment_of(c, w.y, cell_bits, bucket_base);
        }
        order[seg_start[b] + rank[i]] = i;
    }
}

// Probability screening without reading the pair (same argument as sdm_fused.cuh, with bounds over the WHOLE state instead
// of the cell): gamma = 0 whenever the pair's uniform u >= P >= p, where P bounds Eq. 3 through the largest multiplicity
// and the largest volume anywhere in the state (Ctrl::xi_max, Ctrl::v_max_bits) and the cell's own n_s.  A first-in-pair
// droplet whose top uniform word exceeds the threshold leads a pair that provably does nothing: its xi and v -- a 32-byte
// sector each for an 8-byte value in shuffled storage -- are never gathered.  Results are identical (tested with
// SDM_OPT_SCREENING = 0).
struct ScreenBound {
    float v_ub, xi_ub;
};
__device__ __forceinline__ ScreenBound screen_bound(const Ctrl *ctrl)
{
    ScreenBound b;
    b.v_ub = __double2float_ru(__longlong_as_double((long long)((volatile Ctrl *)ctrl)->v_max_bits));
    b.xi_ub = __ll2float_ru(((volatile Ctrl *)ctrl)->xi_max);
    return b;
}
__device__ __forceinline__ uint32_t screen_threshold(const StepParams &prm, const ScreenBound &b, int n_s)
{
    if (!prm.screening) return 0xFFFFFFFFu;
    const int ratio = (n_s & 1) ? n_s : n_s - 1;
    const float norm_ub = __fmul_ru(prm.dtdv_ub_f, (float)max(ratio, 0));
    return flag_threshold_f(cell_probability_bound_f(prm.kernel, prm.kparam_ub_f, b.v_ub, b.xi_ub, norm_ub));
}

// Rows a4-a6 for the candidate pairs that lie inside one sorted segment [s, s+m) of the cell that
// starts at cs and holds n_s droplets (Fig. 4: positions cs+2k, cs+2k+1 pair up).
// sorted[e] = storage index at position s+e.  A pair whose second member is the first droplet of the
// next segment is left to k_pairs_straddle.  Returns events | zeros << 10 | exact << 20 of this lane.
__device__ __forceinline__ int segment_pairs(const int *sorted, int s, int m, int cs, int n_s, int lane,
                                             int64_t *__restrict__ xi, double *__restrict__ v,
                                             const StepParams &prm, const ScreenBound &sb)
{
    const double norm = pair_norm(n_s, prm.dtdv);
    int packed = 0;
    if (prm.no_pairs) return 0;
    const uint32_t thr = screen_threshold(prm, sb, n_s);
    for (int e = ((s - cs) & 1) + 2 * lane; e + 1 < m; e += 64) {
        const int a = sorted[e], b = sorted[e + 1];
        const uint4 w = droplet_block_any((uint32_t)a, prm.step, prm.rk);
        if (w.w > thr) continue;                          // u >= P >= p: gamma = 0, nothing to read
        const double u = block_uniform(w);
        const int r = collide_pair_exact<true>(xi, v, a, b, u, norm, prm.kernel, prm.kparam, prm.attr);
        packed += (r & 1) + (((r >> 1) & 1) << 10) + (1 << 20);
    }
    return packed;
}

// seg_start[0..n_seg]: segment boundaries in order[]; split != 0: segments are pieces of cells and
// cell_bits[cell] gives the key bits a segment's droplets share.  seg_cap <= 256: larger segments are
// ranked by counting (tests lower it).
template <int E>
__global__ void __launch_bounds__(kGenWarps * 32, 4)      // latency-bound gathers: occupancy over registers
k_segment_sort_pairs(const int *__restrict__ seg_start, int n_seg, int split, int seg_cap,
                     const int *__restrict__ order, const int32_t *__restrict__ cell,
                     const int *__restrict__ cell_bits, const int *__restrict__ cell_start,
                     int *__restrict__ idx, int64_t *__restrict__ xi,
                     double *__restrict__ v, Ctrl *ctrl, const __grid_constant__ StepParams prm)
{
    constexpr int L = 32, N = L * E;                      // segment capacity of this instantiation
    extern __shared__ __align__(1024) unsigned char smem_dyn[];
    GenSmem *sm = reinterpret_cast<GenSmem *>(smem_dyn) + (threadIdx.x >> 5);
    const int lane = lane_id();
    const uint32_t sm_base = smem_addr(sm);
    if ((sm_base & 1023u) != 0u) __trap();
    const PhiloxKey &rk = prm.rk;
    for (int i = lane; i < 256; i += 32) sm->cnt[i] = 0;
    __syncwarp();
    seg_cap = min(seg_cap, N);
    int packed_sum_ev = 0, packed_sum_z = 0, packed_sum_ex = 0;
    const ScreenBound sb = screen_bound(ctrl);
    const int warps_total = gridDim.x * kGenWarps;
    for (int seg = blockIdx.x * kGenWarps + (threadIdx.x >> 5); seg < n_seg; seg += warps_total) {
        const int s = seg_start[seg];
        const int m = seg_start[seg + 1] - s;
        if (m == 0) continue;
        const int id0 = order[s];
        const int c = split ? cell[id0] : seg;            // unsplit: a segment is a cell
        const int cs = cell_start[c], n_s = cell_start[c + 1] - cs;
        int pk;
        if (m > seg_cap) {
            warp_rank_by_counting(order + s, 0, m, s, idx, prm.step, rk, lane);
            __threadfence_block();
            __syncwarp();
            pk = segment_pairs(idx + s, s, m, cs, n_s, lane, xi, v, prm, sb);
        } else if (m == 1) {
            if (lane == 0) idx[s] = id0;
            pk = 0;
        } else {
            const int nrem = m - lane;
            int id[E];
#pragma unroll
            for (int k = 0; k < E; ++k) {
                id[k] = (nrem > L * k) ? order[s + lane + L * k] : 0;
                sm->ids[lane + L * k] = id[k];
            }
            const int shift = split ? cell_bits[c] : 0;
            uint32_t x[E];
            count_sort_ids<E>(id, m, lane, shift, prm.step, rk, sm, sm_base, x);
            // adjacent words that share the truncated key differ by less than N
            const uint32_t nx0 = __shfl_down_sync(0xffffffffu, x[0], 1);
            uint32_t dmin = 0xFFFFFFFFu;
            const int l0 = m - E * lane;                  // position 8*lane + r exists iff r < l0
#pragma unroll
            for (int r = 0; r + 1 < E; ++r)
                if (l0 > r + 1) dmin = min(dmin, x[r + 1] - x[r]);
            if (l0 > E) dmin = min(dmin, nx0 - x[E - 1]);
            if (__any_sync(0xffffffffu, dmin < (uint32_t)N)) {
                // exact path: bitonic network on (key64, storage index), R7
                int P = 2;
                while (P < m) P <<= 1;
                for (int e = lane; e < P; e += 32) {
                    if (e < m) {
                        const int d = sm->ids[e];
                        sm->key()[e] = block_key64(droplet_block_any((uint32_t)d, prm.step, rk));
                        sm->sid[e] = d;
                    } else {
                        sm->key()[e] = ~0ull;
                        sm->sid[e] = 0x7fffffff;
                    }
                }
                __syncwarp();
                warp_bitonic(sm->key(), sm->sid, P, lane);
            } else {
#pragma unroll
                for (int r = 0; r < E; ++r)
                    if (l0 > r) sm->sid[E * lane + r] = sm->ids[x[r] & (N - 1)];
                __syncwarp();
            }
            for (int e = lane; e < m; e += 32) idx[s + e] = sm->sid[e];
            pk = segment_pairs(sm->sid, s, m, cs, n_s, lane, xi, v, prm, sb);
            __syncwarp();                                 // ids[], sid[] and slot[] are rewritten by the next segment
        }
        packed_sum_ev += pk & 1023; packed_sum_z += (pk >> 10) & 1023; packed_sum_ex += pk >> 20;
    }
    const int events = __reduce_add_sync(0xffffffffu, packed_sum_ev);
    const int zeros = __reduce_add_sync(0xffffffffu, packed_sum_z);
    const int exact = __reduce_add_sync(0xffffffffu, packed_sum_ex);
    if (lane == 0) {
        if (events) atomicAdd(&ctrl->n_events, (unsigned long long)events);
        if (zeros) atomicAdd(&ctrl->zero_count, zeros);
        if (exact) atomicAdd(&ctrl->n_exact, (unsigned long long)exact);
    }
}

// Split cells only: the candidate pair whose members are the last droplet of one segment and the first
// of the next segment of the same cell.  One thread per segment boundary.
__global__ void __launch_bounds__(256)
k_pairs_straddle(const int *__restrict__ seg_start, int n_seg, const int *__restrict__ idx,
                 const int32_t *__restrict__ cell, const int *__restrict__ cell_start,
                 int64_t *__restrict__ xi, double *__restrict__ v, Ctrl *ctrl,
                 const __grid_constant__ StepParams prm)
{
    const int n = ctrl->n;
    int events = 0, zeros = 0, exact = 0;
    if (prm.no_pairs) return;
    const ScreenBound sb = screen_bound(ctrl);
    for (int seg = blockIdx.x * blockDim.x + threadIdx.x + 1; seg < n_seg; seg += gridDim.x * blockDim.x) {
        const int p = seg_start[seg];
        if (p >= n || seg_start[seg - 1] == p) continue;   // an empty predecessor: boundary p belongs to an earlier seg
        const int a = idx[p - 1], b = idx[p];
        const int c = cell[a];
        if (cell[b] != c) continue;
        const int cs = cell_start[c];
        if ((p - 1 - cs) & 1) continue;                    // a is a second-in-pair
        const uint4 w = droplet_block_any((uint32_t)a, prm.step, prm.rk);
        if (w.w > screen_threshold(prm, sb, cell_start[c + 1] - cs)) continue;
        const double u = block_uniform(w);
        const int r = collide_pair_exact<true>(xi, v, a, b, u, pair_norm(cell_start[c + 1] - cs, prm.dtdv), prm.kernel,
                                         prm.kparam, prm.attr);
        events += r & 1;
        zeros += (r >> 1) & 1;
        exact += 1;
    }
    events = __reduce_add_sync(0xffffffffu, events);
    zeros = __reduce_add_sync(0xffffffffu, zeros);
    exact = __reduce_add_sync(0xffffffffu, exact);
    if (lane_id() == 0) {
        if (events) atomicAdd(&ctrl->n_events, (unsigned long long)events);
        if (zeros) atomicAdd(&ctrl->zero_count, zeros);
        if (exact) atomicAdd(&ctrl->n_exact, (unsigned long long)exact);
    }
}

}  // namespace sdmk
