// sdm_fused.cuh -- the dominant kernel: one SDM coalescence step on cell-contiguous storage.
//
// A group of L lanes owns one cell (E droplets per lane, cell capacity N = L*E; a warp works on
// 32/L cells at once).  Per cell:
//   1. stream xi, v once (coalesced, evict-first) and reduce an upper bound of the largest
//      multiplicity and volume of the cell -> P_cell, an upper bound of Eq. 3 for EVERY pair the
//      permutation could form in this cell ("screening", below); with MOM the same values feed the
//      moment sums;
//   2. one Philox4x32-10 block per droplet (row a1) -> a packed 32-bit sort word
//      (top key bits | local index) and the smallest top uniform word of the lane;
//   3. register-resident bitonic network over the N packed words: in-lane min/max for strides
//      < E, __shfl_xor for lane strides (row a3); words that tie on the truncated key are put in
//      exact (key64, storage index) order by a rare slow path, so idx is bit-exact;
//   4. idx written as vectors (row a3 output); pairs (2m, 2m+1) sit in one lane (row a4);
//   5. only pairs whose first member is flagged evaluate Eq. 3-6 in fp64 (rows a5-a6), exactly as
//      collide_pair_exact does for every pair on the general path.
//
// Why this shape: the kernel is bound by the integer ALU pipe (min/max of the sorting network, the
// xors of Philox), not by HBM.  A compare-exchange between lanes costs a shuffle and two ALU
// instructions per word, one inside a lane costs one, so cells are given to as few lanes as the
// register file allows.
//
// Screening keeps results bit-identical: gamma = floor(p) + [u < p - floor(p)] is 0 whenever
// p < 1 and u >= p.  P_cell >= p holds for every pair of the cell because K is bounded through the
// monotone bounds R >= r_j and W >= w_j (gravitational) or 2*v_max (Golovin) with explicit
// relative margins (1e-4 .. 1e-6) that dwarf all rounding errors of the exact evaluation, and
// u >= (top 32 bits of u) * 2^-32.  A droplet is flagged iff its top-32-bit uniform <= ceil(P_cell*2^32);
// P_cell >= 1 (or NaN/inf) flags everything.  Unflagged pairs are skipped: they are no-ops.
#pragma once

#include "sdm_kernels.cuh"

namespace sdmk {

constexpr int kFusedWarps = 8;

// Bitonic network over N = L*E words held as x[r] at position (lane_in_group*E + r); every
// compare-exchange puts the minimum at the lower position.  Masks stay below L, so shuffles never
// leave the group.
template <int E, int L>
__device__ __forceinline__ void group_sort_packed(uint32_t (&x)[E], int lane)
{
    constexpr int N = L * E;
#pragma unroll
    for (int k = 2; k <= N; k <<= 1) {
        // first stage of the merge: partner p ^ (k-1)
        if (k <= E) {
#pragma unroll
            for (int r = 0; r < E; ++r) {
                const int q = r ^ (k - 1);
                if (q > r) {
                    uint32_t lo = min(x[r], x[q]), hi = max(x[r], x[q]);
                    x[r] = lo; x[q] = hi;
                }
            }
        } else {
            const int lm = k / E - 1;
            const bool lower = (lane & (k / (2 * E))) == 0;
            uint32_t y[E];
#pragma unroll
            for (int r = 0; r < E; ++r) y[r] = __shfl_xor_sync(0xffffffffu, x[E - 1 - r], lm);
#pragma unroll
            for (int r = 0; r < E; ++r) x[r] = lower ? min(x[r], y[r]) : max(x[r], y[r]);
        }
        // remaining stages: partner p ^ j
#pragma unroll
        for (int j = k >> 2; j > 0; j >>= 1) {
            if (j < E) {
#pragma unroll
                for (int r = 0; r < E; ++r) {
                    if ((r & j) == 0) {
                        uint32_t lo = min(x[r], x[r | j]), hi = max(x[r], x[r | j]);
                        x[r] = lo; x[r | j] = hi;
                    }
                }
            } else {
                const int lm = j / E;
                const bool lower = (lane & lm) == 0;
#pragma unroll
                for (int r = 0; r < E; ++r) {
                    uint32_t y = __shfl_xor_sync(0xffffffffu, x[r], lm);
                    x[r] = lower ? min(x[r], y) : max(x[r], y);
                }
            }
        }
    }
}

// Upper bound of Eq. 3 over all pairs of a cell (see the header of this file).
__device__ __forceinline__ double cell_probability_bound(int32_t ktype, double kparam, double v_ub,
                                                         double xi_ub, double norm)
{
    double K;
    if (ktype == 0) {
        K = kparam * 2.0 * v_ub;                                        // b (v_j + v_k) <= 2 b v_max
    } else {
        const double c = 0x1.e8ec8a4aeacc4p-3, pi = 0x1.921fb54442d18p+1;
        float x32 = __double2float_ru(v_ub * c * 1.000001);
        double R = (double)cbrtf(x32) * 1.0001;                         // cbrtf: <= 1 ulp (fp32)
        R = fmax(R, 1e-12);                                             // raising a bound keeps it a bound
        double W = terminal_velocity(R) * 1.000001;                     // w is non-decreasing in r
        K = kparam * pi * 4.0 * R * R * W;                              // (r_j + r_k)^2 |w_j - w_k| <= 4 R^2 W
    }
    return K * xi_ub * norm * 1.000001;
}

__device__ __forceinline__ uint32_t flag_threshold(double P)
{
    double t = P * 4294967296.0;
    if (!(t < 4294967295.0)) return 0xFFFFFFFFu;                        // P >= 1, inf or NaN: flag all
    return (uint32_t)t + 1u;
}

// Rare: some adjacent sorted words tie on the truncated key.  Re-rank every tie run by the exact
// (key64, local index) order.  sk: this group's N sorted words in shared memory (in/out).
// Works on shared memory only, so that the caller's register arrays never
// get their address taken.  Called by the whole warp (every group with its own cell).
__device__ __noinline__ void fix_key_ties(uint32_t *sk, int E, int N, int s, int n_s, int li, uint64_t seed,
                                          uint32_t base, uint64_t step, const unsigned long long *debug_keys = nullptr)
{
    PhiloxKey rk;
    philox_round_keys(seed, base, rk);
    rk.debug_keys = debug_keys;
    uint32_t mine[32], dst[32];
    for (int r = 0; r < E; ++r) {
        const int p = li * E + r;
        const uint32_t me = sk[p];
        mine[r] = me;
        dst[r] = (uint32_t)p;
        if (p >= n_s) continue;
        int a = p, b = p + 1;
        while (a > 0 && ((sk[a - 1] ^ me) < (uint32_t)N)) --a;
        while (b < n_s && ((sk[b] ^ me) < (uint32_t)N)) ++b;
        if (b - a < 2) continue;
        const int l = (int)(me & (uint32_t)(N - 1));
        const uint64_t key = block_key64(droplet_block_any((uint32_t)(s + l), step, rk));
        int rank = 0;
        for (int q = a; q < b; ++q) {
            if (q == p) continue;
            const int l2 = (int)(sk[q] & (uint32_t)(N - 1));
            const uint64_t key2 = block_key64(droplet_block_any((uint32_t)(s + l2), step, rk));
            rank += key_less(key2, l2, key, l) ? 1 : 0;
        }
        dst[r] = (uint32_t)(a + rank);
    }
    __syncwarp();                                     // everybody has read; now permute in place
    for (int r = 0; r < E; ++r) sk[dst[r]] = mine[r];
    __syncwarp();
}

// One pair's contribution to (M0, M1, M2), products rounded as in k_moments_global.
__device__ __forceinline__ void pair_moments(const int64_t *xi, const double *v, int a, int b, int64_t &p0,
                                             double &p1, double &p2)
{
    const int64_t xa = xi[a], xb = xi[b];
    const double va = v[a], vb = v[b];
    const double ya = __dmul_rn(__ll2double_rn(xa), va), yb = __dmul_rn(__ll2double_rn(xb), vb);
    p0 = xa + xb;
    p1 = __dadd_rn(ya, yb);
    p2 = __dadd_rn(__dmul_rn(ya, va), __dmul_rn(yb, vb));
}

// Rare: the cell has flagged droplets.  Evaluate rows a5-a6 exactly for the pairs they lead.
// sk: the group's sorted words; sflag[k]: ballot word of element slot k (bit = lane of the warp);
// lane0: first lane of the group.  delta (may be NULL): three doubles per lane receiving the change
// of (M0, M1, M2) caused by this lane's events (M0's change as the bit pattern of an int64).
template <bool TAB>
__device__ __noinline__ int collide_flagged(const uint32_t *sk, const uint32_t *sflag, int E, int L, int lane0,
                                            int64_t *xi, double *v, int s, int n_s, int li, double dtdv,
                                            int32_t ktype, double kparam, uint64_t seed, uint32_t base, uint64_t step,
                                            double *delta, const AttrView &av)
{
    const uint32_t N = (uint32_t)(E * L);
    int64_t d0 = 0;
    double d1 = 0.0, d2 = 0.0;
    PhiloxKey rk;
    philox_round_keys(seed, base, rk);
    const double norm = pair_norm(n_s, dtdv);
    int packed = 0;                                   // events | zeros << 10 | exact << 20
    for (int m = 0; m < E / 2; ++m) {
        const int p = li * E + 2 * m;
        if (p + 1 >= n_s) continue;
        const int a = (int)(sk[p] & (N - 1)), b = (int)(sk[p + 1] & (N - 1));
        // droplet a was element slot a / L of lane lane0 + a % L
        if (((sflag[a / L] >> (lane0 + a % L)) & 1u) == 0) continue;
        const double u = block_uniform(droplet_block_any((uint32_t)(s + a), step, rk));
        int64_t o0 = 0;
        double o1 = 0.0, o2 = 0.0;
        if (delta) pair_moments(xi, v, s + a, s + b, o0, o1, o2);
        const int r = collide_pair_exact<TAB>(xi, v, s + a, s + b, u, norm, ktype, kparam, av);
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

// Cells larger than the kernel's capacity cannot reach it (the host checks the largest cell at
// sdm_set_state and cells never grow); this keeps the result defined anyway.  Whole warp, one cell.
template <bool TAB>
__device__ __noinline__ int oversize_cell(int64_t *xi, double *v, int *idx, int s, int n_s, int lane,
                                          double dtdv, int32_t ktype, double kparam, uint64_t seed, uint32_t base,
                                          uint64_t step, double *delta, const AttrView &av,
                                          const unsigned long long *debug_keys = nullptr)
{
    PhiloxKey rk;
    philox_round_keys(seed, base, rk);
    rk.debug_keys = debug_keys;
    warp_rank_by_counting(nullptr, s, n_s, s, idx, step, rk, lane);
    __syncwarp();
    const double norm = pair_norm(n_s, dtdv);
    int packed = 0;
    for (int q = lane; q < (n_s >> 1); q += 32) {
        int a = idx[s + 2 * q], b = idx[s + 2 * q + 1];
        double u = block_uniform(droplet_block_any((uint32_t)a, step, rk));
        int r = collide_pair_exact<TAB>(xi, v, a, b, u, norm, ktype, kparam, av);
        packed += (r & 1) + (((r >> 1) & 1) << 10) + (1 << 20);
    }
    if (delta) {                                      // here: the cell's whole post-step contribution
        __syncwarp();
        int64_t d0 = 0;
        double d1 = 0.0, d2 = 0.0;
        for (int q = lane; q < n_s; q += 32) {
            const int64_t x = xi[s + q];
            const double vol = v[s + q];
            const double xv = __dmul_rn(__ll2double_rn(x), vol);
            d0 += x;
            d1 = __dadd_rn(d1, xv);
            d2 = __dadd_rn(d2, __dmul_rn(xv, vol));
        }
        delta[0] = __longlong_as_double(d0);
        delta[1] = d1;
        delta[2] = d2;
    }
    return packed;
}

template <int E>
struct FusedTraits {
        static constexpr int kMinBlocks = (E >= 16) ? 2 : 3;
};

// MOM: also produce the global moments (M0, M1, M2) of the state AFTER the step: the pre-step sums
// are taken from the values streamed for the screening, and every event adds its exact change.
template <int E, int L, bool MOM, bool TAB>
__global__ void __launch_bounds__(kFusedWarps * 32, FusedTraits<E>::kMinBlocks)
k_fused_cells(int64_t *__restrict__ xi, double *__restrict__ v, const int *__restrict__ cell_start,
              int n_cell, int *__restrict__ idx, Ctrl *ctrl, StepParams prm, int64_t *__restrict__ part0,
              double *__restrict__ part1, double *__restrict__ part2, int64_t *__restrict__ m0,
              double *__restrict__ m1, double *__restrict__ m2)
{
    constexpr int N = L * E;                  // cell capacity
    constexpr int G = 32 / L;                 // cells per warp
    static_assert(E >= 2 && (E & (E - 1)) == 0 && (L & (L - 1)) == 0 && L <= 32, "bad shape");
    __shared__ uint32_t s_scratch[kFusedWarps][G][N];         // rare paths only
    __shared__ uint32_t s_flags[kFusedWarps][E];
    __shared__ double s_delta[MOM ? kFusedWarps * 32 * 3 : 1];
    double *my_delta = MOM ? &s_delta[(threadIdx.x >> 5) * 96 + (threadIdx.x & 31) * 3] : nullptr;
    int64_t a0 = 0;
    double a1 = 0.0, a2 = 0.0;
    const int warp = threadIdx.x >> 5, lane = lane_id();
    const int g = lane / L, li = lane % L, lane0 = g * L;
    PhiloxKey rk;
    philox_round_keys(prm.seed, prm.rk.base, rk);
    rk.debug_keys = prm.rk.debug_keys;
    int events = 0, zeros = 0, exact = 0;
    const int cells_per_round = gridDim.x * kFusedWarps * G;
    for (int cbase = (blockIdx.x * kFusedWarps + warp) * G; cbase < n_cell; cbase += cells_per_round) {
        const int c = cbase + g;
        int s = 0, n_s = 0;
        if (c < n_cell) {
            s = cell_start[c];
            n_s = cell_start[c + 1] - s;
        }
        if (__any_sync(0xffffffffu, n_s > N)) {
            for (int gg = 0; gg < G; ++gg) {
                const int s2 = __shfl_sync(0xffffffffu, s, gg * L), n2 = __shfl_sync(0xffffffffu, n_s, gg * L);
                if (n2 <= N) continue;
                const int pk = oversize_cell<TAB>(xi, v, idx, s2, n2, lane, prm.dtdv, prm.kernel, prm.kparam,
                                             prm.seed, prm.rk.base, prm.step, my_delta, prm.attr, prm.rk.debug_keys);
                events += pk & 1023; zeros += (pk >> 10) & 1023; exact += pk >> 20;
                if (MOM) {
                    a0 += __double_as_longlong(my_delta[0]);
                    a1 = __dadd_rn(a1, my_delta[1]);
                    a2 = __dadd_rn(a2, my_delta[2]);
                }
                __syncwarp();
            }
            if (n_s > N) n_s = 0;                 // done
        }
        // 1. stream the cell once: bounds of max xi and max v (volumes are positive doubles, so the
        //    high word orders them; multiplicities are rounded up to fp32); moment sums with MOM
        uint32_t vhi_max = 0;
        float xi_max = 0.0f;
        const int nrem = n_s - li;                        // droplet k*L+li exists iff nrem > k*L
        if (prm.screening || MOM) {
            const long long *px = reinterpret_cast<const long long *>(xi + s + li);
            const double *pv = v + s + li;
#pragma unroll
            for (int k = 0; k < E; ++k) {
                const int64_t lx = (nrem > L * k) ? __ldcs(px + L * k) : 0;
                const double lv = (nrem > L * k) ? __ldcs(pv + L * k) : 0.0;
                vhi_max = max(vhi_max, (uint32_t)__double2hiint(lv));
                xi_max = fmaxf(xi_max, __ll2float_ru(lx));
                if (MOM) {                                  // absent droplets were loaded as (0, 0.0)
                    const double xv = __dmul_rn(__ll2double_rn(lx), lv);
                    a0 += lx;
                    a1 = __dadd_rn(a1, xv);
                    a2 = __dadd_rn(a2, __dmul_rn(xv, lv));
                }
            }
#pragma unroll
            for (int d = 1; d < L; d <<= 1) {
                vhi_max = max(vhi_max, __shfl_xor_sync(0xffffffffu, vhi_max, d));
                xi_max = fmaxf(xi_max, __shfl_xor_sync(0xffffffffu, xi_max, d));
            }
        }
        uint32_t thr = 0xFFFFFFFFu;
        if (prm.screening) {
            const double v_ub = __hiloint2double((int)(vhi_max + 1u), 0);
            const double P = cell_probability_bound(prm.kernel, prm.kparam_ub, v_ub, (double)xi_max,
                                                    pair_norm(n_s, prm.dtdv));
            thr = flag_threshold(P);
        }
        // 2. Philox block per droplet -> packed sort word; smallest top uniform word of the lane
        uint32_t x[E];
        uint32_t umin = 0xFFFFFFFFu;
        const uint32_t sid0 = (uint32_t)(s + li);
#pragma unroll
        for (int k = 0; k < E; ++k) {
            const uint4 w = droplet_block_any(sid0 + (uint32_t)(L * k), prm.step, rk);
            const bool valid = nrem > L * k;
            x[k] = valid ? ((w.y & ~(uint32_t)(N - 1)) | (uint32_t)(li + L * k)) : 0xFFFFFFFFu;
            umin = min(umin, valid ? w.w : 0xFFFFFFFFu);
        }
        // 3. sort, then exact order inside truncated-key ties (rare)
        group_sort_packed<E, L>(x, lane);
        {
            // words that share the truncated key differ by less than N (necessary, not sufficient:
            // the slow path re-checks); sorted ascending, so differences are non-negative
            // (sentinel words behind the last droplet are all equal and excluded: position li*E + r exists iff r < l0)
            const uint32_t nx = __shfl_down_sync(0xffffffffu, x[0], 1);
            const int l0 = n_s - E * li;
            uint32_t dmin = (li < L - 1 && l0 > E) ? nx - x[E - 1] : 0xFFFFFFFFu;
#pragma unroll
            for (int r = 0; r + 1 < E; ++r)
                if (l0 > r + 1) dmin = min(dmin, x[r + 1] - x[r]);
            if (__any_sync(0xffffffffu, dmin < (uint32_t)N)) {
                uint32_t *sk = s_scratch[warp][g];
#pragma unroll
                for (int r = 0; r < E; ++r) sk[li * E + r] = x[r];
                __syncwarp();
                fix_key_ties(sk, E, N, s, n_s, li, prm.seed, prm.rk.base, prm.step, prm.rk.debug_keys);
#pragma unroll
                for (int r = 0; r < E; ++r) x[r] = sk[li * E + r];
                __syncwarp();
            }
        }
        // 4. idx
        if (prm.write_idx) {
            const int p0 = li * E;
            if (((s & (N - 1)) == 0) && (E % 4 == 0) && (p0 + E <= n_s)) {
                // cell start aligned to the capacity: s + local == s | local
#pragma unroll
                for (int r = 0; r < E; r += 4) {
                    int4 o = make_int4(s | (int)(x[r] & (N - 1)), s | (int)(x[r + 1] & (N - 1)),
                                       s | (int)(x[r + 2] & (N - 1)), s | (int)(x[r + 3] & (N - 1)));
                    __stcs(reinterpret_cast<int4 *>(idx + s + p0 + r), o);
                }
            } else if (((s & 3) == 0) && (E % 4 == 0) && (p0 + E <= n_s)) {
#pragma unroll
                for (int r = 0; r < E; r += 4) {
                    int4 o = make_int4(s + (int)(x[r] & (N - 1)), s + (int)(x[r + 1] & (N - 1)),
                                       s + (int)(x[r + 2] & (N - 1)), s + (int)(x[r + 3] & (N - 1)));
                    __stcs(reinterpret_cast<int4 *>(idx + s + p0 + r), o);
                }
            } else {
#pragma unroll
                for (int r = 0; r < E; ++r)
                    if (p0 + r < n_s) idx[s + p0 + r] = s + (int)(x[r] & (N - 1));
            }
        }
        // 5. pairs led by a flagged droplet (rare)
        if (__any_sync(0xffffffffu, umin <= thr)) {
            // redo the blocks of this lane's droplets to learn which ones are flagged
#pragma unroll 1
            for (int k = 0; k < E; ++k) {
                const uint4 w = droplet_block_any(sid0 + (uint32_t)(L * k), prm.step, rk);
                const uint32_t word = __ballot_sync(0xffffffffu, (nrem > L * k) && (w.w <= thr));
                if (lane == (k & 31)) s_flags[warp][k] = word;
            }
            uint32_t *sk = s_scratch[warp][g];
#pragma unroll
            for (int r = 0; r < E; ++r) sk[li * E + r] = x[r];
            __syncwarp();
            const int pk = collide_flagged<TAB>(sk, s_flags[warp], E, L, lane0, xi, v, s, n_s, li, prm.dtdv,
                                           prm.kernel, prm.kparam, prm.seed, prm.rk.base, prm.step, my_delta, prm.attr);
            events += pk & 1023; zeros += (pk >> 10) & 1023; exact += pk >> 20;
            if (MOM) {
                a0 += __double_as_longlong(my_delta[0]);
                a1 = __dadd_rn(a1, my_delta[1]);
                a2 = __dadd_rn(a2, my_delta[2]);
            }
            __syncwarp();
        }
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
