// sdm_box.cuh -- the single-cell box path (BASELINE.json configs 1-3: n_cell == 1, 2^13 .. 2^20 droplets): ALL steps of
// an sdm_run, or one sdm_coalescence_step, in ONE cooperative launch of a persistent grid.
//
// A box is one cell, so row a3 is a global sort of n (key64, storage index) pairs every step, and the general path
// spends it in seven dependent launches (count / scan / scatter / segment sort / straddling pairs ...), each at the
// launch-latency floor for the smaller boxes.  Here the grid of G CTAs (G <= number of SMs, all co-resident) keeps
// running and meets at two grid-wide barriers per step:
//
//   A1  CTA c takes the storage indices of its chunk [c*ch, (c+1)*ch): one Philox block per droplet (row a1; nothing
//       is read from memory), destination region d = floor(key_hi * G / 2^32) (keys are uniform, so regions fill
//       evenly, and d is monotone in the key: the sorted order is region 0, region 1, ...), histogram of d in shared
//       memory, then ONE returning atomic per (c, d) on the region totals: the returned value is where c's records
//       start inside region d.
//   --- barrier 1 ---   (zeros to remove? rare: the grid runs the stable compaction pass, then repeats A1)
//   A2  every CTA scans the G region totals -> region offsets; the 8-byte records (key_hi, index) are written to their
//       place in the record queue (L2-resident): a counting sort by region without a single per-droplet global atomic.
//   --- barrier 2 ---
//   B   CTA d sorts region d in shared memory -- counting sort on sub-buckets of ~8 records, rank inside the sub-bucket
//       by counting, exact (key_lo, index) order inside key_hi ties by re-evaluating Philox -- writes its slice of
//       idx, and evaluates rows a4-a6 for the pairs (2m, 2m+1) of the GLOBAL order that start in its slice; a pair that
//       straddles two regions takes its second member from the first sorted record the neighbour publishes.
//
// Phase A of step t+1 touches no state (only indices and n), and the queue and the region totals are double-buffered,
// so B(t) of a slow CTA may overlap A(t+1) of a fast one; barrier 2 of step t+1 orders B(t) before B(t+1).
// Results are those of the per-step general path bit for bit (same Philox stream, same order, same pair arithmetic:
// collide_pair_exact).  Regions larger than the shared-memory capacity (more than 20 sigma above the mean for every
// size the host admits) are ranked by counting in global memory: slow, but defined for every input.
#pragma once

#include "sdm_general.cuh"

#ifndef SDM_MAX_ATTR
#define SDM_MAX_ATTR 8
#endif

namespace sdmk {

constexpr int kBoxThreads = 1024;
constexpr int kBoxMaxCtas = 255;            // G <= min(SM count, this): a region number fits 8 bits
constexpr int kBoxChunkMax = 8192;          // storage indices per CTA in phase A (records staged in shared memory)
constexpr int kBoxMeanMax = 7800;           // the host admits n <= G * this: mean + 12 sigma + 32 <= kBoxRegionMax
constexpr int kBoxRegionMax = 9216;         // records per region that phase B sorts in shared memory
constexpr int kBoxSubMax = 2048;            // sub-buckets of a region

struct BoxCtrl {                            // in the workspace; zeroed before every launch
    unsigned int bar;                       // grid barrier: arrivals since launch
    unsigned int overflow[3];               // some region exceeded its fixed capacity (by step mod 3)
    int coltot[3][kBoxMaxCtas + 1];         // records per region, by step mod 3: written in phase A of step t, read after
                                            // the barrier of step t, cleared after the barrier of step t+1, reused at t+3
    unsigned long long first_rec[2][kBoxMaxCtas + 1];   // first sorted record of region d (step parity)
    unsigned int first_tag[2][kBoxMaxCtas + 1];         // local step number + 1 of the record above
};

struct BoxSmem {
    // phase A: records and (region, rank) of this CTA's chunk; phase B: the region, twice, and the sub-bucket table
    unsigned long long rec0[kBoxRegionMax]; // A: records of the chunk          B: records grouped by sub-bucket
    unsigned long long rec1[kBoxRegionMax]; //                                  B: sorted records
    uint32_t aux[kBoxRegionMax];            // A: region | rank << 8            B: sub-bucket | rank << 11
    int cnt2[kBoxSubMax];                   // A: histogram / base of regions   B: sub-bucket counts
    int start2[kBoxSubMax + 1];             // A: region offsets                B: sub-bucket starts
    int warp_tot[33];
    int scalar[4];
};
// the rare in-launch compaction (8 warps) runs while phase A's staging is void: its tile buffers alias rec0 .. aux
static_assert(sizeof(CompactSmem) + (size_t)(SDM_MAX_ATTR - 1) * kCompactTile * 8 <=
                  2 * sizeof(unsigned long long) * kBoxRegionMax + sizeof(uint32_t) * kBoxRegionMax,
              "compaction buffers must fit into the record buffers");

constexpr size_t kBoxSmemBytes = sizeof(BoxSmem);

// grid-wide barrier of a cooperative launch (all CTAs resident): monotone arrival counter, release/acquire through
// __threadfence (which also drops stale L1 lines, as cooperative_groups' grid sync relies on)
// `after_acquire` runs in thread 0 only, between the acquire fence and the closing CTA barrier: the place to read a
// global flag ONCE per CTA and publish it in shared memory, so that all threads of the CTA branch on the same value
// (a flag that another CTA clears later must not be re-read by a slow warp: it would take a different path to the
// next barrier).
template <class F>
__device__ __forceinline__ void box_grid_sync(BoxCtrl *box, unsigned int G, unsigned int &epoch, F after_acquire)
{
    __syncthreads();
    epoch += 1;
    if (threadIdx.x == 0) {
        __threadfence();
        atomicAdd(&box->bar, 1u);
        const unsigned int target = epoch * G;
        while (*((volatile unsigned int *)&box->bar) < target) { }
        __threadfence();
        after_acquire();
    }
    __syncthreads();
}
__device__ __forceinline__ void box_grid_sync(BoxCtrl *box, unsigned int G, unsigned int &epoch)
{
    box_grid_sync(box, G, epoch, [] {});
}

// exclusive scan of v[0..m) in shared memory by the whole CTA (m <= 2 * blockDim); out[m] = total
__device__ __forceinline__ void box_block_scan(const int *v, int *out, int m, int *warp_tot)
{
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int i0 = 2 * tid, a = i0 < m ? v[i0] : 0, b = i0 + 1 < m ? v[i0 + 1] : 0;
    int inc = a + b;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += t;
    }
    if (lane == 31) warp_tot[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        const int w = warp_tot[lane];
        int winc = w;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, winc, d);
            if (lane >= d) winc += t;
        }
        warp_tot[lane] = winc - w;
        if (lane == 31) warp_tot[32] = winc;
    }
    __syncthreads();
    const int excl = warp_tot[warp] + inc - (a + b);
    if (i0 < m) out[i0] = excl;
    if (i0 + 1 < m) out[i0 + 1] = excl + a;
    if (tid == 0) out[m] = warp_tot[32];
    __syncthreads();
}

// exact order of two records (R7): key_hi, then key_lo (re-evaluated), then storage index
__device__ __forceinline__ bool box_less_exact(unsigned long long a, unsigned long long b, uint64_t step, const PhiloxKey &rk)
{
    const uint32_t ha = (uint32_t)(a >> 32), hb = (uint32_t)(b >> 32);
    if (ha != hb) return ha < hb;
    const uint32_t ia = (uint32_t)a, ib = (uint32_t)b;
    const uint32_t la = droplet_block_any(ia, step, rk).x, lb = droplet_block_any(ib, step, rk).x;
    return la < lb || (la == lb && ia < ib);
}

__global__ void __launch_bounds__(kBoxThreads, 1)
k_box_steps(int64_t *__restrict__ xi, double *__restrict__ v, int32_t *__restrict__ cell, int *__restrict__ idx,
            int *__restrict__ cell_start, Ctrl *ctrl, BoxCtrl *box, unsigned long long *__restrict__ queue,
            long long queue_stride, int region_cap, int sort_cap, unsigned long long *__restrict__ tile_status, int n_steps,
            int remove_zero,
            const __grid_constant__ StepParams prm)
{
    extern __shared__ __align__(16) unsigned char box_smem_raw[];
    BoxSmem &sm = *reinterpret_cast<BoxSmem *>(box_smem_raw);
    CompactSmem &csm = *reinterpret_cast<CompactSmem *>(box_smem_raw);          // aliases rec0 .. (see above)
    double *s_extra = reinterpret_cast<double *>(box_smem_raw + ((sizeof(CompactSmem) + 15) & ~(size_t)15));
    const int tid = threadIdx.x, c = blockIdx.x;
    const unsigned int G = gridDim.x;
    const PhiloxKey &rk = prm.rk;
    unsigned int epoch = 0;
    int events = 0, exact = 0;
    int n = ((volatile Ctrl *)ctrl)->n;             // changes only in the in-launch compaction, which re-reads it
    for (int t = 0; t < n_steps; ++t) {
        const uint64_t step = prm.step + (uint64_t)t;
        const int p = t & 1, pc = t % 3;
        unsigned long long *q = queue + (long long)p * queue_stride;
        int m_src, lo;
        bool exact_layout = false;    // false: region d of the queue starts at d * region_cap; true: at its exact offset
        // ---------------- A: Philox, region histogram, records to the queue ----------------
        while (true) {
            const int ch = (n + (int)G - 1) / (int)G;
            lo = min(n, c * ch);
            m_src = min(n, lo + ch) - lo;
            for (int d = tid; d < (int)G; d += kBoxThreads) sm.cnt2[d] = 0;
            __syncthreads();
            if (m_src > kBoxChunkMax) __trap();           // the host admits n <= G * kBoxChunkMax, and n never grows
            for (int e = tid; e < m_src; e += kBoxThreads) {
                const uint32_t i = (uint32_t)(lo + e);
                const uint4 w = droplet_block_any(i, step, rk);
                const uint32_t d = __umulhi(w.y, G);
                const int r = atomicAdd(&sm.cnt2[d], 1);
                sm.rec0[e] = ((unsigned long long)w.y << 32) | i;
                sm.aux[e] = d | ((uint32_t)r << 8);
            }
            __syncthreads();
            for (int d = tid; d < (int)G; d += kBoxThreads) {
                const int k = sm.cnt2[d];
                const int r0 = k ? atomicAdd(&box->coltot[pc][d], k) : 0;    // where this chunk's records start in region d
                sm.cnt2[d] = r0;
                if (!exact_layout && r0 + k > region_cap) atomicOr(&box->overflow[pc], 1u);
            }
            if (!exact_layout) {
                // fast layout: fixed-capacity regions (mean + 12 sigma), so the records can leave now and the step
                // needs ONE grid barrier; an overflowing region (never with Philox keys) falls back to exact offsets
                __syncthreads();
                for (int e = tid; e < m_src; e += kBoxThreads) {
                    const uint32_t a = sm.aux[e], d = a & 255u;
                    const int pos = sm.cnt2[d] + (int)(a >> 8);
                    if (pos < region_cap) q[(long long)d * region_cap + pos] = sm.rec0[e];
                }
            }
            // ---- every B of the previous step is complete; totals are final.  Thread 0 reads the two flags that decide
            // the CTA's path once and publishes them: the last CTA to finish a compaction clears zero_count, and CTA 0
            // clears the overflow flag, while a slow warp of another CTA may not have branched yet.
            box_grid_sync(box, G, epoch, [&] {
                sm.scalar[1] = remove_zero ? ((volatile Ctrl *)ctrl)->zero_count : 0;
                sm.scalar[2] = (int)((volatile unsigned int *)box->overflow)[pc];
            });
            const int zeros_seen = sm.scalar[1], overflow_seen = sm.scalar[2];
            if (zeros_seen != 0) {
                // rare: step 0 of Fig. 3 inside the launch -- the stable compaction pass (warps 0-7), then phase A again
                if (tid < kCompactThreads)
                    compact_tiles(xi, v, cell, ctrl, tile_status, prm.attr, csm, s_extra, tid, G,
                                  [] { asm volatile("bar.sync 1, %0;" :: "n"(kCompactThreads) : "memory"); });
                box_grid_sync(box, G, epoch);
                if (c == 0) {
                    for (int d = tid; d < (int)G; d += kBoxThreads) box->coltot[pc][d] = 0;
                    if (tid == 0) box->overflow[pc] = 0u;
                }
                box_grid_sync(box, G, epoch);
                n = ((volatile Ctrl *)ctrl)->n;
                continue;
            }
            if (!exact_layout && overflow_seen != 0) {
                box_grid_sync(box, G, epoch);             // everybody has seen the flag
                if (c == 0) {
                    for (int d = tid; d < (int)G; d += kBoxThreads) box->coltot[pc][d] = 0;
                    if (tid == 0) box->overflow[pc] = 0u;
                }
                box_grid_sync(box, G, epoch);
                exact_layout = true;
                continue;
            }
            break;
        }
        // region offsets in the sorted order: exclusive scan of the region totals
        for (int d = tid; d < (int)G; d += kBoxThreads) sm.start2[d] = ((volatile int *)box->coltot[pc])[d];
        __syncthreads();
        if (tid < 32) {                                   // G <= 255: one warp, 8 totals per lane
            int loc[8], sum = 0;
#pragma unroll
            for (int k = 0; k < 8; ++k) { const int d = tid * 8 + k; loc[k] = d < (int)G ? sm.start2[d] : 0; sum += loc[k]; }
            int inc = sum;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int u = __shfl_up_sync(0xffffffffu, inc, d);
                if (tid >= d) inc += u;
            }
            int run = inc - sum;
#pragma unroll
            for (int k = 0; k < 8; ++k) { const int d = tid * 8 + k; if (d <= (int)G) sm.start2[d] = run; run += loc[k]; }
        }
        __syncthreads();
        const int my_off = sm.start2[c], m = sm.start2[c + 1] - my_off;
        int next_nonempty = -1;                           // the first region after this one that holds a record
        if (tid == 0) {
            for (int d = c + 1; d < (int)G; ++d)
                if (sm.start2[d + 1] > sm.start2[d]) { next_nonempty = d; break; }
            sm.scalar[0] = next_nonempty;
        }
        if (exact_layout) {                               // exact offsets: the records leave now, second barrier
            for (int e = tid; e < m_src; e += kBoxThreads) {
                const uint32_t a = sm.aux[e], d = a & 255u, r = a >> 8;
                q[sm.start2[d] + sm.cnt2[d] + (int)r] = sm.rec0[e];
            }
            box_grid_sync(box, G, epoch);
        } else {
            __syncthreads();
        }
        next_nonempty = sm.scalar[0];
        if (c == 0) {                                     // the totals of step t-1: everybody has read them (see BoxCtrl)
            for (int d = tid; d < (int)G; d += kBoxThreads) box->coltot[(t + 2) % 3][d] = 0;
        }
        // ---------------- B: sort region c, idx, pairs ----------------
        const unsigned long long *qr = exact_layout ? q + my_off : q + (long long)c * region_cap;
        const double norm = pair_norm(n, prm.dtdv);
        if (m > sort_cap) {
            // never with Philox keys (> 20 sigma); defined anyway: rank by counting in global memory
            for (int e = tid; e < m; e += kBoxThreads) {
                const unsigned long long me = __ldcg(qr + e);
                int rank = 0;
                for (int f = 0; f < m; ++f) {
                    const unsigned long long o = __ldcg(qr + f);
                    if (f != e && box_less_exact(o, me, step, rk)) ++rank;
                }
                idx[my_off + rank] = (int)(uint32_t)me;
                if (rank == 0) {
                    ((volatile unsigned long long *)box->first_rec[p])[c] = me;
                    __threadfence();
                    ((volatile unsigned int *)box->first_tag[p])[c] = (unsigned int)t + 1u;
                }
            }
            __threadfence();
            __syncthreads();
        } else if (m > 0) {
            // sub-buckets of ~3 records (at most 2048 of them): j = floor((key_hi - first key of the region) * S / width), monotone in the key
            const int S = max(1, min(kBoxSubMax, (m + 2) / 3));
            const unsigned long long kb0 = (((unsigned long long)c << 32) + G - 1) / G;
            const unsigned long long kb1 = (((unsigned long long)(c + 1) << 32) + G - 1) / G;
            const unsigned long long M = ((unsigned long long)S << 32) / (kb1 - kb0);
            auto sub_of = [&](unsigned long long rec) -> int {
                return (int)((((rec >> 32) - kb0) * M) >> 32);
            };
            for (int j = tid; j < S; j += kBoxThreads) sm.cnt2[j] = 0;
            __syncthreads();
            for (int e = tid; e < m; e += kBoxThreads) {
                const unsigned long long rec = __ldcg(qr + e);
                const int j = sub_of(rec);
                const int r = atomicAdd(&sm.cnt2[j], 1);
                sm.rec1[e] = rec;
                sm.aux[e] = (uint32_t)j | ((uint32_t)r << 11);
            }
            __syncthreads();
            box_block_scan(sm.cnt2, sm.start2, S, sm.warp_tot);
            for (int e = tid; e < m; e += kBoxThreads) {
                const uint32_t a = sm.aux[e];
                sm.rec0[sm.start2[a & 2047u] + (int)(a >> 11)] = sm.rec1[e];
            }
            __syncthreads();
            // rank inside the sub-bucket by counting on (key_hi, index)
            for (int e = tid; e < m; e += kBoxThreads) {
                const unsigned long long me = sm.rec0[e];
                const int j = sub_of(me), a = sm.start2[j], b = sm.start2[j + 1];
                int rank = 0;
                for (int f = a; f < b; ++f) rank += sm.rec0[f] < me ? 1 : 0;
                sm.rec1[a + rank] = me;
            }
            __syncthreads();
            // exact order inside runs of equal key_hi (about one pair per region and step at 2^20 droplets)
            for (int e = tid; e < m; e += kBoxThreads) {
                const unsigned long long me = sm.rec1[e];
                const uint32_t h = (uint32_t)(me >> 32);
                int dst = e;
                const bool tl = e > 0 && (uint32_t)(sm.rec1[e - 1] >> 32) == h;
                const bool tr = e + 1 < m && (uint32_t)(sm.rec1[e + 1] >> 32) == h;
                if (tl || tr) {
                    int a = e, b = e + 1;
                    while (a > 0 && (uint32_t)(sm.rec1[a - 1] >> 32) == h) --a;
                    while (b < m && (uint32_t)(sm.rec1[b] >> 32) == h) ++b;
                    int rank = 0;
                    for (int f = a; f < b; ++f)
                        if (f != e && box_less_exact(sm.rec1[f], me, step, rk)) ++rank;
                    dst = a + rank;
                }
                sm.rec0[dst] = me;
            }
            __syncthreads();
            if (tid == 0) {                               // for the neighbour whose last pair straddles into this region
                ((volatile unsigned long long *)box->first_rec[p])[c] = sm.rec0[0];
                __threadfence();
                ((volatile unsigned int *)box->first_tag[p])[c] = (unsigned int)t + 1u;
            }
            for (int e = tid; e < m; e += kBoxThreads) idx[my_off + e] = (int)(uint32_t)sm.rec0[e];
        }
        // rows a4-a6: pairs (2k, 2k+1) of the global order whose first member lies in this region; the loads of a
        // thread's next pair are issued before the arithmetic of the current one (L2 gathers: one round trip in all)
        if (m > 0 && !prm.no_pairs) {
            const bool big = m > sort_cap;
            if (big) __threadfence();
            // state-wide probability screening (sdm_general.cuh): a first-in-pair droplet whose top uniform word exceeds
            // the threshold leads a pair with gamma = 0 -- nothing of it is read
            const uint32_t thr = screen_threshold(prm, screen_bound(ctrl), n);
            // the next pair at or after position e (stride 2 * kBoxThreads) that passes the screening
            auto next_pair = [&](int &e, int &a, int &b, uint4 &w) -> bool {
                for (; e < m && my_off + e + 1 < n; e += 2 * kBoxThreads) {
                    a = big ? ((volatile int *)idx)[my_off + e] : (int)(uint32_t)sm.rec0[e];
                    w = droplet_block_any((uint32_t)a, step, rk);
                    if (w.w > thr) continue;
                    if (e + 1 < m) {
                        b = big ? ((volatile int *)idx)[my_off + e + 1] : (int)(uint32_t)sm.rec0[e + 1];
                    } else {
                        while (((volatile unsigned int *)box->first_tag[p])[next_nonempty] != (unsigned int)t + 1u) { }
                        __threadfence();
                        b = (int)(uint32_t)((volatile unsigned long long *)box->first_rec[p])[next_nonempty];
                    }
                    return true;
                }
                return false;
            };
            int e = tid * 2 + (my_off & 1), a = 0, b = 0;
            uint4 w = make_uint4(0u, 0u, 0u, 0u);
            bool have = next_pair(e, a, b, w);
            int64_t xa = 0, xb = 0;
            double va = 0.0, vb = 0.0;
            if (have) { xa = xi[a]; xb = xi[b]; va = v[a]; vb = v[b]; }
            while (have) {
                e += 2 * kBoxThreads;
                int a2 = 0, b2 = 0;
                uint4 w2 = make_uint4(0u, 0u, 0u, 0u);
                const bool have2 = next_pair(e, a2, b2, w2);
                int64_t xa2 = 0, xb2 = 0;
                double va2 = 0.0, vb2 = 0.0;
                if (have2) { xa2 = xi[a2]; xb2 = xi[b2]; va2 = v[a2]; vb2 = v[b2]; }
                const int r = collide_pair_loaded<true>(xi, v, a, b, xa, xb, va, vb, block_uniform(w), norm, prm.kernel,
                                                        prm.kparam, prm.attr);
                events += r & 1; exact += 1;
                if (r & 2) atomicAdd(&ctrl->zero_count, 1);   // rare; seen by the barrier of the next step
                have = have2; a = a2; b = b2; w = w2; xa = xa2; xb = xb2; va = va2; vb = vb2;
            }
        }
        if (c == 0 && tid == 0) { cell_start[0] = 0; cell_start[1] = n; }
        __syncthreads();                                  // shared memory is rewritten by phase A of the next step
    }
    events = __reduce_add_sync(0xffffffffu, events);
    exact = __reduce_add_sync(0xffffffffu, exact);
    if ((tid & 31) == 0) {
        if (events) atomicAdd(&ctrl->n_events, (unsigned long long)events);
        if (exact) atomicAdd(&ctrl->n_exact, (unsigned long long)exact);
    }
}

}  // namespace sdmk
