// sdm_fused_bucket.cuh -- the dominant kernel for cells of up to 256 droplets on cell-contiguous
// storage: one warp per cell, per-cell permutation by a BUCKET SORT on the (uniform) Philox keys.
//
// The register bitonic network of sdm_fused.cuh costs O(n log^2 n) compare-exchanges and made the
// kernel integer-ALU bound.  Philox keys are uniform, so a counting sort on the top
// 10 key bits puts every droplet within a few places of its final position in O(n):
//   A. one Philox4x32-10 block per droplet (row a1) -> packed 32-bit word (top 24 key bits | local
//      index); shared-memory atomic on a byte-packed histogram of the top 10 key bits;
//   B. warp scan of the 1024 byte counters -> bucket starts (one byte per bucket);
//   C. a second atomic on the start bytes hands every droplet a slot of its bucket's range: slot[]
//      is now sorted by bucket, in arrival order inside a bucket;
//   D. position-centric exact ranking.  Left neighbours belong to the same or a lower bucket, right
//      neighbours to the same or a higher one, so with every bucket <= 4 droplets
//          final position = p - #{d = 1..3 : slot[p-d] > slot[p]} + #{d = 1..3 : slot[p+d] < slot[p]}
//      with no bucket test at all; a lane ranks 4 consecutive positions from three 16-byte loads.
//      Cells with a larger bucket (0.7 %) rank by a loop over the bucket (bucket_rank_slow);
//   E. lanes read their sorted quads; from here on the kernel is the one of sdm_fused.cuh: exact
//      re-ranking of truncated-key ties, idx as 16-byte stores, screening, flagged pairs.
// A byte counter that overflows (a bucket of >= 256 droplets, or any carry) makes the scanned total
// differ from n_s: the cell then ranks its words by plain counting (never happens with Philox keys;
// SDM_OPT_SORT_FALLBACK forces it for the tests).  Results equal the plain argsort by (key64, storage index) bit for bit.
#pragma once

#include "sdm_fused.cuh"

namespace sdmk {

constexpr int kBucketWarps = 8;
constexpr int kBucketCap = 256;           // cell capacity of this kernel
constexpr int kBucketRows = 8;            // droplets per lane
constexpr int kBucketBits = 10;           // key bits of the counting sort (1024 buckets, mean occupancy 1/4)
constexpr int kBucketWords = (1 << kBucketBits) / 4;
constexpr int kBucketWindow = 3;          // neighbours inspected on each side in phase D

struct __align__(16) BucketSmem {
    uint32_t cnt[kBucketWords];           // byte counters (zero between cells)
    uint32_t start[kBucketWords];         // byte bucket starts, then running fill positions
    uint32_t pad_lo[4];                   // zeros: "no larger word to the left"
    uint32_t slot[kBucketCap];            // words grouped by bucket, arrival order inside
    uint32_t pad_hi[4];                   // ones: "no smaller word to the right"
    uint32_t sorted[kBucketCap];          // words in final order
};

// Positions of all words by counting (O(n^2) shared-memory reads): the defined result for any
// histogram overflow.  In: slot[l] = word of droplet l.  Out: sorted[].
__device__ __noinline__ void bucket_sort_fallback(BucketSmem *sm, int n_s, int lane)
{
    for (int p = lane; p < kBucketCap; p += 32) sm->sorted[p] = 0xFFFFFFFFu;
    __syncwarp();
    for (int l = lane; l < n_s; l += 32) {
        const uint32_t me = sm->slot[l];
        int rank = 0;
        for (int q = 0; q < n_s; ++q) rank += (sm->slot[q] < me) ? 1 : 0;   // words are distinct
        sm->sorted[rank] = me;
    }
    __syncwarp();
}

// Phase D for cells with a bucket larger than the window allows: same rule, the scan runs to the
// ends of the bucket.  slot[] (with sentinels past n_s) -> sorted[].
__device__ __noinline__ void bucket_rank_slow(BucketSmem *sm, int lane)
{
    for (int p = lane; p < kBucketCap; p += 32) {
        const uint32_t me = sm->slot[p], b = me >> (32 - kBucketBits);
        int pos = p;
        for (int q = p - 1; q >= 0; --q) {
            const uint32_t o = sm->slot[q];
            if ((o >> (32 - kBucketBits)) != b) break;
            pos -= (o > me) ? 1 : 0;
        }
        for (int q = p + 1; q < kBucketCap; ++q) {
            const uint32_t o = sm->slot[q];
            if ((o >> (32 - kBucketBits)) != b) break;
            pos += (o < me) ? 1 : 0;
        }
        sm->sorted[pos] = me;
    }
}

// q += d where o > me / o < me, as a compare and ONE predicated add (the compiler's own choice is a
// three-instruction select)
__device__ __forceinline__ void add_if_gt(int &q, uint32_t o, uint32_t me, int d)
{
    asm("{\n\t.reg .pred p;\n\tsetp.gt.u32 p, %1, %2;\n\t@p add.s32 %0, %0, %3;\n\t}" : "+r"(q) : "r"(o), "r"(me), "r"(d));
}
// both words of an in-quad pair move when the later one (b, position qb) is the smaller
__device__ __forceinline__ void swap_if_lt(int &qa, int &qb, uint32_t a, uint32_t b)
{
    asm("{\n\t.reg .pred p;\n\tsetp.lt.u32 p, %3, %2;\n\t@p add.s32 %0, %0, 1;\n\t@p add.s32 %1, %1, -1;\n\t}"
        : "+r"(qa), "+r"(qb) : "r"(a), "r"(b));
}

// Rank the four words of one quad (a) given the quads before (l) and after (r) it; p = position of a.x.
// Window of three neighbours on each side.
__device__ __forceinline__ void rank_quad(const uint4 l, const uint4 a, const uint4 r, int p, uint32_t *sorted)
{
    int q0 = p, q1 = p + 1, q2 = p + 2, q3 = p + 3;
    swap_if_lt(q0, q1, a.x, a.y);
    swap_if_lt(q0, q2, a.x, a.z);
    swap_if_lt(q0, q3, a.x, a.w);
    swap_if_lt(q1, q2, a.y, a.z);
    swap_if_lt(q1, q3, a.y, a.w);
    swap_if_lt(q2, q3, a.z, a.w);
    // to the left larger words move us down, to the right smaller words move us up
    add_if_gt(q0, l.y, a.x, -1); add_if_gt(q0, l.z, a.x, -1); add_if_gt(q0, l.w, a.x, -1);
    add_if_gt(q1, l.z, a.y, -1); add_if_gt(q1, l.w, a.y, -1);
    add_if_gt(q2, l.w, a.z, -1);
    add_if_gt(q1, a.y, r.x, 1);
    add_if_gt(q2, a.z, r.x, 1); add_if_gt(q2, a.z, r.y, 1);
    add_if_gt(q3, a.w, r.x, 1); add_if_gt(q3, a.w, r.y, 1); add_if_gt(q3, a.w, r.z, 1);
    sorted[q0] = a.x;
    sorted[q1] = a.y;
    sorted[q2] = a.z;
    sorted[q3] = a.w;
}

// Rows a5-a6 for the pairs led by a flagged droplet (rare).  Lane owns positions 4*lane..4*lane+3 and
// 128+4*lane..; sflag[k]: ballot word of droplet row k (bit = lane).  See collide_flagged.
__device__ __noinline__ int collide_flagged_quads(const uint32_t *sk, const uint32_t *sflag, int64_t *xi,
                                                  double *v, int s, int n_s, int lane, double dtdv,
                                                  int32_t ktype, double kparam, uint64_t seed, uint64_t step,
                                                  double *delta)
{
    int64_t d0 = 0;
    double d1 = 0.0, d2 = 0.0;
    PhiloxKey rk;
    philox_round_keys(seed, rk);
    const double norm = pair_norm(n_s, dtdv);
    int packed = 0;                                   // events | zeros << 10 | exact << 20
    for (int m = 0; m < 4; ++m) {
        const int p = (m >> 1) * 128 + 4 * lane + 2 * (m & 1);
        if (p + 1 >= n_s) continue;
        const int a = (int)(sk[p] & 255u), b = (int)(sk[p + 1] & 255u);
        if (((sflag[a >> 5] >> (a & 31)) & 1u) == 0) continue;
        const double u = block_uniform(droplet_block((uint32_t)(s + a), step, rk));
        int64_t o0 = 0;
        double o1 = 0.0, o2 = 0.0;
        if (delta) pair_moments(xi, v, s + a, s + b, o0, o1, o2);
        const int r = collide_pair_exact(xi, v, s + a, s + b, u, norm, ktype, kparam);
        if (delta && (r & 1)) {
            int64_t n0;
            double n1, n2;
            pair_moments(xi, v, s + a, s + b, n0, n1, n2);
            d0 += n0 - o0;
            d1 = __dadd_rn(d1, __dsub_rn(n1, o1));
            d2 = __dadd_rn(d2, __dsub_rn(n2, o2));
        }
        packed += (r & 1) + (((r >> 1) & 1) << 10) + (1 << 20);
    }
    if (delta) {
        delta[0] = __longlong_as_double(d0);
        delta[1] = d1;
        delta[2] = d2;
    }
    return packed;
}

template <bool MOM>
__global__ void __launch_bounds__(kBucketWarps * 32, 3)
k_fused_cells_bucket(int64_t *__restrict__ xi, double *__restrict__ v, const int *__restrict__ cell_start,
                     int n_cell, int *__restrict__ idx, Ctrl *ctrl, StepParams prm,
                     int64_t *__restrict__ part0, double *__restrict__ part1, double *__restrict__ part2,
                     int64_t *__restrict__ m0, double *__restrict__ m1, double *__restrict__ m2)
{
    constexpr int N = kBucketCap, E = kBucketRows, L = 32;
    __shared__ BucketSmem s_b[kBucketWarps];
    __shared__ uint32_t s_flags[kBucketWarps][E];
    __shared__ double s_delta[MOM ? kBucketWarps * 32 * 3 : 1];
    double *my_delta = MOM ? &s_delta[(threadIdx.x >> 5) * 96 + (threadIdx.x & 31) * 3] : nullptr;
    int64_t a0 = 0;
    double a1 = 0.0, a2 = 0.0;
    const int warp = threadIdx.x >> 5, lane = lane_id();
    BucketSmem *sm = &s_b[warp];
    PhiloxKey rk;
    philox_round_keys(prm.seed, rk);
    int events = 0, zeros = 0, exact = 0;
    for (int i = lane; i < kBucketWords; i += 32) sm->cnt[i] = 0;
    if (lane < 4) { sm->pad_lo[lane] = 0u; sm->pad_hi[lane] = 0xFFFFFFFFu; }
    __syncwarp();
    const int cells_per_round = gridDim.x * kBucketWarps;
    for (int c = blockIdx.x * kBucketWarps + warp; c < n_cell; c += cells_per_round) {
        const int s = cell_start[c];
        const int n_s = cell_start[c + 1] - s;
        if (n_s > N) {                                        // cannot happen (host checks); defined anyway
            const int pk = oversize_cell(xi, v, idx, s, n_s, lane, prm.dtdv, prm.kernel, prm.kparam, prm.seed,
                                         prm.step, my_delta);
            events += pk & 1023; zeros += (pk >> 10) & 1023; exact += pk >> 20;
            if (MOM) {
                a0 += __double_as_longlong(my_delta[0]);
                a1 = __dadd_rn(a1, my_delta[1]);
                a2 = __dadd_rn(a2, my_delta[2]);
            }
            __syncwarp();
            continue;
        }
        // 1. stream the cell once: bounds of max xi and max v for the screening; moment sums with MOM
        uint32_t vhi_max = 0;
        float xi_max = 0.0f;
        const int nrem = n_s - lane;                          // droplet k*32+lane exists iff nrem > 32k
        if (prm.screening || MOM) {
            const long long *px = reinterpret_cast<const long long *>(xi + s + lane);
            const double *pv = v + s + lane;
#pragma unroll
            for (int k = 0; k < E; ++k) {
                const int64_t lx = (nrem > L * k) ? __ldcs(px + L * k) : 0;
                const double lv = (nrem > L * k) ? __ldcs(pv + L * k) : 0.0;
                vhi_max = max(vhi_max, (uint32_t)__double2hiint(lv));
                xi_max = fmaxf(xi_max, __ll2float_ru(lx));
                if (MOM) {
                    const double xv = __dmul_rn(__ll2double_rn(lx), lv);
                    a0 += lx;
                    a1 = __dadd_rn(a1, xv);
                    a2 = __dadd_rn(a2, __dmul_rn(xv, lv));
                }
            }
            vhi_max = __reduce_max_sync(0xffffffffu, vhi_max);
            xi_max = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(xi_max)));   // xi_max >= 0
        }
        uint32_t thr = 0xFFFFFFFFu;
        if (prm.screening) {
            const double v_ub = __hiloint2double((int)(vhi_max + 1u), 0);
            const double P = cell_probability_bound(prm.kernel, prm.kparam, v_ub, (double)xi_max,
                                                    pair_norm(n_s, prm.dtdv));
            thr = flag_threshold(P);
        }
        // A. Philox block per droplet -> packed word; bucket histogram
        uint32_t xw[E];
        uint32_t umin = 0xFFFFFFFFu;
        const uint32_t sid0 = (uint32_t)(s + lane);
#pragma unroll
        for (int k = 0; k < E; ++k) {
            const uint4 w = droplet_block(sid0 + (uint32_t)(L * k), prm.step, rk);
            const bool valid = nrem > L * k;
            xw[k] = valid ? ((w.y & ~(uint32_t)(N - 1)) | (uint32_t)(lane + L * k)) : 0xFFFFFFFFu;
            umin = min(umin, valid ? w.w : 0xFFFFFFFFu);
        }
#pragma unroll
        for (int k = 0; k < E; ++k) {
            if (nrem > L * k) {
                const uint32_t b = xw[k] >> (32 - kBucketBits);
                atomicAdd(&sm->cnt[b >> 2], 1u << ((b & 3u) << 3));
            }
        }
        __syncwarp();
        // B. scan of the byte counters (lane owns kBucketWords/32 consecutive words)
        constexpr int WPL = kBucketWords / 32;
        uint32_t cw[WPL], pw[WPL];
#pragma unroll
        for (int i = 0; i < WPL; i += 4) {
            const uint4 q = reinterpret_cast<const uint4 *>(sm->cnt)[(lane * WPL + i) >> 2];
            cw[i] = q.x; cw[i + 1] = q.y; cw[i + 2] = q.z; cw[i + 3] = q.w;
            reinterpret_cast<uint4 *>(sm->cnt)[(lane * WPL + i) >> 2] = make_uint4(0u, 0u, 0u, 0u);
        }
        uint32_t tot = 0, cmax = 0;
#pragma unroll
        for (int i = 0; i < WPL; ++i) {
            pw[i] = cw[i] * 0x01010101u;                      // inclusive byte prefix sums inside the word
            cmax = __vmaxu4(cmax, cw[i]);
            const uint32_t t = pw[i] >> 24;
            pw[i] = (pw[i] - cw[i]) + tot * 0x01010101u;      // exclusive, relative to the lane's first bucket
            tot += t;
        }
        uint32_t inc = tot;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, inc, d);
            if (lane >= d) inc += t;
        }
        const uint32_t excl = (inc - tot) * 0x01010101u;
        const bool overflow = (__shfl_sync(0xffffffffu, inc, 31) != (uint32_t)n_s) || prm.sort_fallback;
        if (!overflow) {
            // starts past the last droplet may wrap (value 256): those buckets are empty, never read
#pragma unroll
            for (int i = 0; i < WPL; i += 4)
                reinterpret_cast<uint4 *>(sm->start)[(lane * WPL + i) >> 2] =
                    make_uint4(pw[i] + excl, pw[i + 1] + excl, pw[i + 2] + excl, pw[i + 3] + excl);
            const bool big = __any_sync(0xffffffffu,
                                        __vcmpgtu4(cmax, 0x01010101u * (uint32_t)(kBucketWindow + 1)) != 0u);
            __syncwarp();
            // C. the start bytes become fill pointers: a second atomic hands out the slots of a bucket
            //    (sentinels behind the last droplet).  A bucket ending at 256 wraps its byte and carries
            //    into the next bucket, which is then empty like all later ones.
#pragma unroll
            for (int k = 0; k < E; ++k) {
                if (nrem > L * k) {
                    const uint32_t b = xw[k] >> (32 - kBucketBits), sh = (b & 3u) << 3;
                    const uint32_t old = atomicAdd(&sm->start[b >> 2], 1u << sh);
                    sm->slot[(old >> sh) & 0xFFu] = xw[k];
                } else if (n_s < N) {
                    sm->slot[L * k + lane] = 0xFFFFFFFFu;
                }
            }
            __syncwarp();
            // D. exact positions
            if (!big) {
                const uint4 *q4 = reinterpret_cast<const uint4 *>(sm->pad_lo);      // quad j is q4[j + 1]
#pragma unroll
                for (int k = 0; k < 2; ++k) {
                    const int j = k * 32 + lane;
                    rank_quad(q4[j], q4[j + 1], q4[j + 2], 4 * j, sm->sorted);
                }
            } else {
                bucket_rank_slow(sm, lane);
            }
            __syncwarp();
        } else {
            __syncwarp();
#pragma unroll
            for (int k = 0; k < E; ++k) sm->slot[L * k + lane] = xw[k];
            __syncwarp();
            bucket_sort_fallback(sm, n_s, lane);
        }
        // E. sorted words of positions 4*lane .. 4*lane+3 and 128+4*lane .. 128+4*lane+3
        uint32_t x[E];
        {
            const uint4 q0 = reinterpret_cast<const uint4 *>(sm->sorted)[lane];
            const uint4 q1 = reinterpret_cast<const uint4 *>(sm->sorted)[32 + lane];
            x[0] = q0.x; x[1] = q0.y; x[2] = q0.z; x[3] = q0.w;
            x[4] = q1.x; x[5] = q1.y; x[6] = q1.z; x[7] = q1.w;
        }
        {
            // words that share the truncated key differ by less than N; exact order by the slow path.
            // The successor of a quad's last word is the first word of the next quad.
            const uint32_t f0 = __shfl_down_sync(0xffffffffu, x[0], 1), f1 = __shfl_down_sync(0xffffffffu, x[4], 1);
            const uint32_t w0 = __shfl_sync(0xffffffffu, x[4], 0);
            const uint32_t n0 = (lane < 31) ? f0 : w0;
            uint32_t dmin = 0xFFFFFFFFu;
            if (n_s == N) {
                dmin = min(min(x[1] - x[0], x[2] - x[1]), min(x[3] - x[2], n0 - x[3]));
                dmin = min(dmin, min(min(x[5] - x[4], x[6] - x[5]), x[7] - x[6]));
                if (lane < 31) dmin = min(dmin, f1 - x[7]);
            } else {                                          // the padding words are all equal: skip them
                const int l0 = n_s - 4 * lane, l1 = l0 - 128; // position 4*lane + r exists iff r < l0
                if (l0 > 1) dmin = min(dmin, x[1] - x[0]);
                if (l0 > 2) dmin = min(dmin, x[2] - x[1]);
                if (l0 > 3) dmin = min(dmin, x[3] - x[2]);
                if (l0 > 4) dmin = min(dmin, n0 - x[3]);
                if (l1 > 1) dmin = min(dmin, x[5] - x[4]);
                if (l1 > 2) dmin = min(dmin, x[6] - x[5]);
                if (l1 > 3) dmin = min(dmin, x[7] - x[6]);
                if (l1 > 4) dmin = min(dmin, f1 - x[7]);
            }
            if (__any_sync(0xffffffffu, dmin < (uint32_t)N)) {
                fix_key_ties(sm->sorted, E, N, s, n_s, lane, prm.seed, prm.step);
                const uint4 q0 = reinterpret_cast<const uint4 *>(sm->sorted)[lane];
                const uint4 q1 = reinterpret_cast<const uint4 *>(sm->sorted)[32 + lane];
                x[0] = q0.x; x[1] = q0.y; x[2] = q0.z; x[3] = q0.w;
                x[4] = q1.x; x[5] = q1.y; x[6] = q1.z; x[7] = q1.w;
            }
        }
        // idx (row a3 output): a warp store covers 512 contiguous bytes
        if (prm.write_idx) {
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                const int p = k * 128 + 4 * lane;
                if (((s & 3) == 0) && (p + 4 <= n_s)) {
                    int4 o = make_int4(s + (int)(x[4 * k] & (N - 1)), s + (int)(x[4 * k + 1] & (N - 1)),
                                       s + (int)(x[4 * k + 2] & (N - 1)), s + (int)(x[4 * k + 3] & (N - 1)));
                    __stcs(reinterpret_cast<int4 *>(idx + s + p), o);
                } else {
#pragma unroll
                    for (int r = 0; r < 4; ++r)
                        if (p + r < n_s) idx[s + p + r] = s + (int)(x[4 * k + r] & (N - 1));
                }
            }
        }
        // pairs led by a flagged droplet (rare): rows a5-a6 exactly
        if (__any_sync(0xffffffffu, umin <= thr)) {
#pragma unroll 1
            for (int k = 0; k < E; ++k) {
                const uint4 w = droplet_block(sid0 + (uint32_t)(L * k), prm.step, rk);
                const uint32_t word = __ballot_sync(0xffffffffu, (nrem > L * k) && (w.w <= thr));
                if (lane == k) s_flags[warp][k] = word;
            }
            __syncwarp();
            const int pk = collide_flagged_quads(sm->sorted, s_flags[warp], xi, v, s, n_s, lane, prm.dtdv,
                                                 prm.kernel, prm.kparam, prm.seed, prm.step, my_delta);
            events += pk & 1023; zeros += (pk >> 10) & 1023; exact += pk >> 20;
            if (MOM) {
                a0 += __double_as_longlong(my_delta[0]);
                a1 = __dadd_rn(a1, my_delta[1]);
                a2 = __dadd_rn(a2, my_delta[2]);
            }
        }
        __syncwarp();                                         // sorted[] is rewritten by the next cell
    }
    events = __reduce_add_sync(0xffffffffu, events);
    zeros = __reduce_add_sync(0xffffffffu, zeros);
    exact = __reduce_add_sync(0xffffffffu, exact);
    if (lane == 0) {
        if (events) atomicAdd(&ctrl->n_events, (unsigned long long)events);
        if (zeros) atomicAdd(&ctrl->zero_count, zeros);
        if (exact) atomicAdd(&ctrl->n_exact, (unsigned long long)exact);
    }
    if (MOM) moments_finish(a0, a1, a2, ctrl, part0, part1, part2, m0, m1, m2);
}

}  // namespace sdmk
