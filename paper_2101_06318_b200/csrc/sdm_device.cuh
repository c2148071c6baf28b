// sdm_device.cuh -- device-side arithmetic of the SDM coalescence step (sm_100a).
//
// Every floating-point operation whose result reaches the state is written with an explicit
// round-to-nearest intrinsic (__dmul_rn, __dadd_rn, ...): those are never contracted into FMAs,
// so the results are bit-identical to a plain IEEE-754 evaluation in the same order (the library
// is also compiled with -fmad=false).  Citations: PAPER.md = arXiv 2101.06318; R* = DESIGN.md.
#pragma once

// This header is also compiled at run time by NVRTC (sdm_set_kernel_source: the pair kernel around user-supplied kernel
// code, sdm_user_pairs.cuh), where the toolkit headers are not available.
#ifdef __CUDACC_RTC__
typedef signed int int32_t;
typedef unsigned int uint32_t;
typedef long long int64_t;
typedef unsigned long long uint64_t;
#else
#include <cstdint>
#include <cuda_runtime.h>
#endif

namespace sdmk {

// ---------------------------------------------------------------------------------------------
// Row a1: Philox4x32-10, one block per droplet per step (R6).
// ---------------------------------------------------------------------------------------------
struct PhiloxKey {          // the ten round keys, precomputed once per thread (uniform values)
    uint32_t k0[10], k1[10];
    uint32_t base;          // storage index of the handle's droplet 0 in the GLOBAL state (sdm_set_index_base): the
                            // Philox counter is base + local index, so a shard reproduces the unsharded stream
    const unsigned long long *debug_keys;   // sdm_debug_permutation: sort keys supplied by the caller (by local storage
                                            // index) instead of Philox words 0-1; NULL in every real step
};

__host__ __device__ __forceinline__ void philox_round_keys(uint64_t seed, uint32_t base, PhiloxKey &rk)
{
    rk.base = base;
    rk.debug_keys = nullptr;
    uint32_t a = (uint32_t)seed, b = (uint32_t)(seed >> 32);
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        rk.k0[r] = a;
        rk.k1[r] = b;
        a += 0x9E3779B9u;
        b += 0xBB67AE85u;
    }
}

__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               const PhiloxKey &rk)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        // one 32x32->64 multiply per product (IMAD.WIDE.U32) instead of separate hi and lo halves
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ rk.k0[r];
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ rk.k1[r];
        c0 = n0; c1 = (uint32_t)p1; c2 = n2; c3 = (uint32_t)p0;
    }
    return make_uint4(c0, c1, c2, c3);
}

// counter = {global storage index lo, hi, step lo, hi}; global index = base + local index < 2^32 (checked by
// sdm_set_index_base), so the hi word is 0
__device__ __forceinline__ uint4 droplet_block_global(uint32_t gsid, uint64_t step, const PhiloxKey &rk)
{
    return philox4x32_10(gsid, 0u, (uint32_t)step, (uint32_t)(step >> 32), rk);
}
__device__ __forceinline__ uint4 droplet_block(uint32_t sid, uint64_t step, const PhiloxKey &rk)
{
    return droplet_block_global(sid + rk.base, step, rk);
}

// The same, or -- in sdm_debug_permutation -- the caller's key in words 0-1 and a uniform of (almost) one.  Used by
// every kernel except the fast section of k_fused_cells_count (which such a call does not enter).
__device__ __forceinline__ uint4 droplet_block_any(uint32_t sid, uint64_t step, const PhiloxKey &rk)
{
    if (rk.debug_keys) {
        const unsigned long long k = rk.debug_keys[sid];
        return make_uint4((uint32_t)k, (uint32_t)(k >> 32), 0xFFFFFFFFu, 0xFFFFFFFFu);
    }
    return droplet_block(sid, step, rk);
}

__device__ __forceinline__ uint64_t block_key64(const uint4 &w)
{
    return (uint64_t)w.x | ((uint64_t)w.y << 32);
}

// phi ~ U[0,1): top 53 bits of words 2-3, times 2^-53 (R6)
__device__ __forceinline__ double block_uniform(const uint4 &w)
{
    uint64_t bits = (uint64_t)w.z | ((uint64_t)w.w << 32);
    return __dmul_rn(__ull2double_rn(bits >> 11), 0x1.0p-53);
}

// ---------------------------------------------------------------------------------------------
// Row a5: coalescence kernels (R9, R10) and Eq. 3.
// ---------------------------------------------------------------------------------------------
// Extensive attributes other than the volume: rows 1..N_ATTR-1
// of the paper's 2-D row-major attribute block, row r at p + r*stride.  They never enter Eq. 3; only a pair
// with gamma_tilde > 0 touches them.
struct AttrView {
    double *p;
    long long stride;
    int n;                  // number of extra rows (0: volume is the only attribute)
    // NEXT-2 rides in the same per-pair bundle: the user's collection-efficiency table of
    // SDM_KERNEL_GRAVITATIONAL_TABULATED (R16): eff_tab[eff_n][eff_n] on the radius grid eff_grid[eff_n]
    int eff_n;
    const double *eff_grid;
    const double *eff_tab;
    const double *user_params;   // SDM_KERNEL_USER: the caller's parameter array (device), sdm_set_kernel_source
    unsigned long long *v_max;   // Ctrl::v_max_bits: bit pattern of the largest volume in the state (screening bound of the
                                 // general and box paths); raised by every event that produces a larger volume
};

struct StepParams {
    double dtdv;      // dt / dV, one IEEE division on the host
    double kparam;    // Golovin b, or gravitational E
    double kparam_ub; // upper bound of kparam times the efficiency table's maximum (screening bounds only)
    int32_t kernel;   // SDM_KERNEL_*
    int32_t write_idx;
    uint64_t seed, step;
    int32_t screening;      // 1: per-cell probability screening (sdm_fused.cuh); 0: every pair in fp64
    float dtdv_ub_f;        // dt/dV and kparam_ub rounded UP to fp32 on the host (screening bounds only)
    float kparam_ub_f;
    int32_t no_pairs;       // 1: rows a1-a3 only (the permutation); the caller evaluates the pairs (SDM_KERNEL_USER)
    AttrView attr;          // extra extensive attributes
    PhiloxKey rk;           // round keys of `seed`: kernels that take the parameters as __grid_constant__ read
                            // them straight from the constant bank instead of holding 20 registers
};

// R10: cube root as a fixed sequence of IEEE double operations (no division, no FMA).
__device__ __forceinline__ double cbrt_spec(double x)
{
    uint64_t bits = (uint64_t)__double_as_longlong(x);
    double y = __longlong_as_double((long long)(0x553EEEEEEEEEF000ull - bits / 3ull));
    const double c43 = 0x1.5555555555555p+0, c13 = 0x1.5555555555555p-2;
#pragma unroll
    for (int it = 0; it < 4; ++it) {
        double t = __dmul_rn(y, y);
        t = __dmul_rn(t, y);
        t = __dmul_rn(x, t);
        t = __dmul_rn(c13, t);
        t = __dsub_rn(c43, t);
        y = __dmul_rn(y, t);
    }
    double r = __dmul_rn(__dmul_rn(x, y), y);
    double d = __dsub_rn(__dmul_rn(__dmul_rn(r, r), r), x);
    double h = __dmul_rn(__dmul_rn(y, y), c13);
    return __dsub_rn(r, __dmul_rn(d, h));
}

__device__ __forceinline__ double terminal_velocity(double r)
{
    if (r < 40e-6) return __dmul_rn(__dmul_rn(1.19e8, r), r);
    if (r < 600e-6) return __dmul_rn(8e3, r);
    return __dmul_rn(220.0, __dsqrt_rn(r));
}

// R16: bilinear interpolation of the efficiency table, clamped outside the grid; every operation rounded
__device__ __forceinline__ void efficiency_locate(const double *__restrict__ grid, int n, double r, int &i, double &t)
{
    if (r < grid[0]) { i = 0; t = 0.0; return; }
    if (r >= grid[n - 1]) { i = n - 2; t = 1.0; return; }
    int lo = 0, hi = n - 1;                                             // grid[lo] <= r < grid[hi]
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (grid[mid] <= r) lo = mid; else hi = mid;
    }
    i = lo;
    t = __ddiv_rn(__dsub_rn(r, grid[lo]), __dsub_rn(grid[lo + 1], grid[lo]));
}

__device__ __forceinline__ double collection_efficiency(const AttrView &av, double rj, double rk)
{
    int i, k;
    double t, u;
    efficiency_locate(av.eff_grid, av.eff_n, rj, i, t);
    efficiency_locate(av.eff_grid, av.eff_n, rk, k, u);
    const double *row0 = av.eff_tab + (long long)i * av.eff_n + k, *row1 = row0 + av.eff_n;
    const double e00 = row0[0], e01 = row0[1], e10 = row1[0], e11 = row1[1];
    const double e0 = __dadd_rn(e00, __dmul_rn(t, __dsub_rn(e10, e00)));
    const double e1 = __dadd_rn(e01, __dmul_rn(t, __dsub_rn(e11, e01)));
    return __dadd_rn(e0, __dmul_rn(u, __dsub_rn(e1, e0)));
}

#ifdef SDM_USER_KERNEL
}  // namespace sdmk
// user-supplied kernel code, defined further down in the same run-time translation unit
__device__ double sdm_user_kernel(double vj, double vk, const double *params);
namespace sdmk {
#endif

__device__ __forceinline__ double coalescence_kernel(int32_t type, double kparam, double vj, double vk)
{
    if (type == 0) return __dmul_rn(kparam, __dadd_rn(vj, vk));       // Golovin
    const double c = 0x1.e8ec8a4aeacc4p-3;                              // 3/(4 pi)
    const double pi = 0x1.921fb54442d18p+1;
    double rj = cbrt_spec(__dmul_rn(vj, c));
    double rk = cbrt_spec(__dmul_rn(vk, c));
    double wj = terminal_velocity(rj), wk = terminal_velocity(rk);
    double s = __dadd_rn(rj, rk);
    double K = __dmul_rn(kparam, pi);
    K = __dmul_rn(K, __dmul_rn(s, s));
    return __dmul_rn(K, fabs(__dsub_rn(wj, wk)));
}

// NEXT-2, SDM_KERNEL_GRAVITATIONAL_TABULATED: the gravitational kernel with E = kparam * Etab(r_j, r_k).
__device__ __noinline__ double coalescence_kernel_tabulated(double kparam, double vj, double vk, const AttrView &av)
{
    const double c = 0x1.e8ec8a4aeacc4p-3;                              // 3/(4 pi)
    const double pi = 0x1.921fb54442d18p+1;
    double rj = cbrt_spec(__dmul_rn(vj, c));
    double rk = cbrt_spec(__dmul_rn(vk, c));
    double wj = terminal_velocity(rj), wk = terminal_velocity(rk);
    double s = __dadd_rn(rj, rk);
    double K = __dmul_rn(__dmul_rn(kparam, collection_efficiency(av, rj, rk)), pi);
    K = __dmul_rn(K, __dmul_rn(s, s));
    return __dmul_rn(K, fabs(__dsub_rn(wj, wk)));
}

// [(n^2-n)/2] / floor(n/2) is the exact integer n-1 (n even) or n (n odd) (R2), so the quotient
// of the paper's Eq. 3 needs no division.
__device__ __forceinline__ double pair_norm(int n_s, double dtdv)
{
    int ratio = (n_s & 1) ? n_s : n_s - 1;
    return __dmul_rn(dtdv, (double)ratio);
}

// ---------------------------------------------------------------------------------------------
// Rows a5-a6 for one candidate pair (a = first-in-pair, b = second), in place in global memory.
// Returns bit 0: an event happened (gamma_tilde > 0); bit 1: a multiplicity became zero.
// TAB: the kernel type may be SDM_KERNEL_GRAVITATIONAL_TABULATED.  The dominant kernel is instantiated without
// it for the built-in kernels: it runs at its register limit, and the mere presence of the table code in its
// call graph cost 10 % (measured: 0.383 -> 0.421 ms on C5).
// ---------------------------------------------------------------------------------------------
// collide_pair_loaded: the same with the four values of the pair already in registers (callers that overlap the
// loads of their next pair with the arithmetic of this one).
template <bool TAB>
__device__ __forceinline__ int collide_pair_loaded(int64_t *__restrict__ xi, double *__restrict__ v,
                                                   int a, int b, int64_t xa, int64_t xb, double vj, double vk,
                                                   double u, double norm, int32_t ktype, double kparam,
                                                   const AttrView &av)
{
    int j = a, k = b;
    int64_t xj = xa, xk = xb;
    if (xa < xb) {                                       // PAPER.md:257-259 (strict <, R8)
        j = b; k = a; xj = xb; xk = xa;
        const double t = vj; vj = vk; vk = t;
    }
    if (xk == 0) return 0;                               // R11
#ifdef SDM_USER_KERNEL
    double K = sdm_user_kernel(vj, vk, av.user_params);     // SDM_KERNEL_USER: the only kernel of this translation unit
#else
    double K = (TAB && ktype == 2) ? coalescence_kernel_tabulated(kparam, vj, vk, av)
                                   : coalescence_kernel(ktype, kparam, vj, vk);
#endif
    double p = __dmul_rn(__dmul_rn(K, __ll2double_rn(xj)), norm);      // Eq. 3 in routine order (R3)
#ifdef SDM_USER_KERNEL
    if (!(p > 0.0)) return 0;                            // R20: user code returned a negative value or NaN: no event
#endif
    double fl = floor(p);
    double gamma = (u < __dsub_rn(p, fl)) ? __dadd_rn(fl, 1.0) : fl;       // PAPER.md:102, R4
    if (gamma == 0.0) return 0;                          // gamma_tilde = min(0, q) = 0: the usual case, no division
    int64_t q = xj / xk;
    int64_t g;
    if (fl >= __ll2double_rn(q)) {
        g = q;                                           // cap reached without converting p (R8)
    } else {
        int64_t gi = __double2ll_rz(gamma);
        g = gi < q ? gi : q;                             // Eq. 4
    }
    if (g == 0) return 0;
    int64_t new_n = xj - g * xk;
    const double gd = __ll2double_rn(g);
    double gv = __dmul_rn(gd, vj);
    double vnew = __dadd_rn(vk, gv);                     // both branches produce v_k + g v_j
    {                                                    // keep the state-wide volume bound valid (rarely a new maximum)
        const unsigned long long nb = (unsigned long long)__double_as_longlong(vnew);
        if (nb > *(volatile unsigned long long *)av.v_max) atomicMax(av.v_max, nb);
    }
    if (new_n > 0) {                                     // Eq. 5
        xi[j] = new_n;
        v[k] = vnew;
        for (int r = 0; r < av.n; ++r) {                 // every extensive attribute
            double *A = av.p + (long long)r * av.stride;
            A[k] = __dadd_rn(A[k], __dmul_rn(gd, A[j]));
        }
        return 1;
    }
    int64_t half = xk >> 1;                              // Eq. 6, xk > 0
    xi[j] = half;
    xi[k] = xk - half;
    v[j] = vnew;
    v[k] = vnew;
    for (int r = 0; r < av.n; ++r) {
        double *A = av.p + (long long)r * av.stride;
        const double t = __dadd_rn(A[k], __dmul_rn(gd, A[j]));
        A[j] = t;
        A[k] = t;
    }
    return half == 0 ? 3 : 1;
}

template <bool TAB>
__device__ __forceinline__ int collide_pair_exact(int64_t *__restrict__ xi, double *__restrict__ v,
                                                  int a, int b, double u, double norm,
                                                  int32_t ktype, double kparam, const AttrView &av)
{
    const int64_t xa = xi[a], xb = xi[b];
    const double va = v[a], vb = v[b];                   // four independent loads, one round trip
    return collide_pair_loaded<TAB>(xi, v, a, b, xa, xb, va, vb, u, norm, ktype, kparam, av);
}

}  // namespace sdmk
