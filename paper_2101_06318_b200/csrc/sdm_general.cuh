// sdm_general.cuh -- general path (any storage order, cells of any size): the per-segment sort.
//
// A "segment" is a cell, or -- for cells larger than the warp capacity -- the droplets of a cell whose
// sort key has the same top B bits (sdm_kernels.cuh: split_bits, k_bucket_count, k_scatter).  order[]
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
constexpr int kGenCap = 256;              // segment capacity of the warp counting sort

struct __align__(1024) GenSmem {
    uint32_t cnt[256];                    // histogram in byte units (zero between segments)
    uint32_t start[256];                  // shared-space byte address of each bin's first slot
    uint32_t slot[kGenCap];               // words grouped by bin
    int ids[kGenCap];                     // storage index of local droplet e
    uint64_t key[kGenCap];                // exact path: full keys
    int sid[kGenCap];                     // exact path: indices carried through the network
};
static_assert(sizeof(GenSmem) % 1024 == 0, "GenSmem must tile shared memory in 1 KB units");
static_assert(offsetof(GenSmem, start) == 1024 && offsetof(GenSmem, slot) == 2048, "layout used by the address arithmetic");

constexpr size_t kGenSmemBytes = kGenWarps * sizeof(GenSmem);

// Sort words of one segment: x[k] belongs to local droplet k*32+lane on entry (id[k] its storage index),
// and to sorted position 8*lane+k on return.  shift = key bits shared by the whole segment.
__device__ __forceinline__ void count_sort_ids(const int (&id)[8], int m, int lane, int shift, uint64_t step,
                                               const PhiloxKey &rk, GenSmem *sm, uint32_t sm_base, uint32_t (&x)[8])
{
    constexpr int E = 8, L = 32, N = kGenCap;
    const int nrem = m - lane;
    uint32_t old[E];
#pragma unroll
    for (int k = 0; k < E; ++k) {
        const bool valid = nrem > L * k;
        const uint4 w = droplet_block((uint32_t)id[k], step, rk);
        const uint32_t hi = __funnelshift_l(w.x, w.y, shift);          // top 32 bits of key64 << shift
        x[k] = valid ? ((hi & ~(uint32_t)(N - 1)) | (uint32_t)(lane + L * k)) : 0xFFFFFFFFu;
        old[k] = 0;
        if (valid) old[k] = atoms_add(sm_base | ((hi >> 22) & 0x3FCu), 4u);
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
    {
        const uint4 q0 = reinterpret_cast<const uint4 *>(sm->slot)[2 * lane];
        const uint4 q1 = reinterpret_cast<const uint4 *>(sm->slot)[2 * lane + 1];
        x[0] = q0.x; x[1] = q0.y; x[2] = q0.z; x[3] = q0.w;
        x[4] = q1.x; x[5] = q1.y; x[6] = q1.z; x[7] = q1.w;
    }
    for (uint32_t r = 0; r < rounds; r += 2) {
        cex(x[0], x[1]); cex(x[2], x[3]); cex(x[4], x[5]); cex(x[6], x[7]);
        uint32_t nx0 = __shfl_down_sync(0xffffffffu, x[0], 1);
        uint32_t px7 = __shfl_up_sync(0xffffffffu, x[7], 1);
        if (lane == 31) nx0 = 0xFFFFFFFFu;
        if (lane == 0) px7 = 0u;
        cex(x[1], x[2]); cex(x[3], x[4]); cex(x[5], x[6]);
        x[7] = min(x[7], nx0);
        x[0] = max(x[0], px7);
    }
}

// seg_start[0..n_seg]: segment boundaries in order[]; n_seg_host < 0: the number of segments is
// ctrl->n_buckets (split mode), and cell_bits[cell] gives the key bits a segment's droplets share.
__global__ void __launch_bounds__(kGenWarps * 32)
k_segment_sort_count(const int *__restrict__ seg_start, const Ctrl *__restrict__ ctrl, int n_seg_host,
                     const int *__restrict__ order, const int32_t *__restrict__ cell,
                     const int *__restrict__ cell_bits, int *__restrict__ idx,
                     const __grid_constant__ StepParams prm)
{
    constexpr int E = 8, L = 32, N = kGenCap;
    extern __shared__ __align__(1024) unsigned char smem_dyn[];
    GenSmem *sm = reinterpret_cast<GenSmem *>(smem_dyn) + (threadIdx.x >> 5);
    const int lane = lane_id();
    const uint32_t sm_base = smem_addr(sm);
    if ((sm_base & 1023u) != 0u) __trap();
    const PhiloxKey &rk = prm.rk;
    for (int i = lane; i < 256; i += 32) sm->cnt[i] = 0;
    __syncwarp();
    const bool split = n_seg_host < 0;
    const int n_seg = split ? ctrl->n_buckets : n_seg_host;
    const int warps_total = gridDim.x * kGenWarps;
    for (int seg = blockIdx.x * kGenWarps + (threadIdx.x >> 5); seg < n_seg; seg += warps_total) {
        const int s = seg_start[seg];
        const int m = seg_start[seg + 1] - s;
        if (m == 0) continue;
        if (m > N) {
            warp_rank_by_counting(order + s, 0, m, s, idx, prm.step, rk, lane);
            continue;
        }
        if (m == 1) {
            if (lane == 0) idx[s] = order[s];
            continue;
        }
        const int nrem = m - lane;
        int id[E];
#pragma unroll
        for (int k = 0; k < E; ++k) {
            id[k] = (nrem > L * k) ? order[s + lane + L * k] : 0;
            sm->ids[lane + L * k] = id[k];
        }
        int shift = 0;
        if (split) shift = cell_bits[cell[__shfl_sync(0xffffffffu, id[0], 0)]];
        uint32_t x[E];
        count_sort_ids(id, m, lane, shift, prm.step, rk, sm, sm_base, x);
        // adjacent words that share the truncated key differ by less than N
        const uint32_t nx0 = __shfl_down_sync(0xffffffffu, x[0], 1);
        uint32_t dmin = 0xFFFFFFFFu;
        const int l0 = m - E * lane;                      // position 8*lane + r exists iff r < l0
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
                    sm->key[e] = block_key64(droplet_block((uint32_t)d, prm.step, rk));
                    sm->sid[e] = d;
                } else {
                    sm->key[e] = ~0ull;
                    sm->sid[e] = 0x7fffffff;
                }
            }
            __syncwarp();
            warp_bitonic(sm->key, sm->sid, P, lane);
            for (int e = lane; e < m; e += 32) idx[s + e] = sm->sid[e];
            __syncwarp();
            continue;
        }
#pragma unroll
        for (int r = 0; r < E; ++r)
            if (l0 > r) idx[s + E * lane + r] = sm->ids[x[r] & (N - 1)];
        __syncwarp();                                     // ids[] and slot[] are rewritten by the next segment
    }
}

}  // namespace sdmk
