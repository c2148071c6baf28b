// sdm_spectrum.cuh -- NEXT-3: the spectrum product of Fig. 6: mass of droplets per unit ln r on a
// grid of bins, smoothed with a centered five-bin running mean (R17).
//
// k_spectrum_bin: one pass over (xi, v) -- 16 B per droplet, HBM-bound for large states.  The bin of a droplet
// is found by binary search on the volume edges held in shared memory (exact comparisons: the decision is the
// same integer on every implementation); sums xi*v are accumulated per CTA in shared memory (fp64 atomics) and
// flushed with one global atomic per non-empty bin and CTA.
// k_spectrum_finish: one CTA: value = sum * rho / V / dlnr, then n_smooth passes of the running mean with the
// window truncated at the ends, summed left to right.
#pragma once

#include "sdm_kernels.cuh"

namespace sdmk {

constexpr int kMaxBins = 1024;            // SDM_MAX_BINS

__global__ void __launch_bounds__(256)
k_spectrum_bin(const int64_t *__restrict__ xi, const double *__restrict__ v, const Ctrl *__restrict__ ctrl,
               int n_bins, const double *__restrict__ edges, double *__restrict__ sums)
{
    __shared__ double s_edges[kMaxBins + 1];
    __shared__ double s_sum[kMaxBins];
    for (int b = threadIdx.x; b <= n_bins; b += blockDim.x) s_edges[b] = edges[b];
    for (int b = threadIdx.x; b < n_bins; b += blockDim.x) s_sum[b] = 0.0;
    __syncthreads();
    const int n = ctrl->n;
    const double lo_edge = s_edges[0], hi_edge = s_edges[n_bins];
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const double vol = __ldcs(v + i);
        const int64_t x = __ldcs(xi + i);
        if (!(vol >= lo_edge) || !(vol < hi_edge)) continue;
        int lo = 0, hi = n_bins;                                  // s_edges[lo] <= vol < s_edges[hi]
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (s_edges[mid] <= vol) lo = mid; else hi = mid;
        }
        atomicAdd(&s_sum[lo], __dmul_rn(__ll2double_rn(x), vol));
    }
    __syncthreads();
    for (int b = threadIdx.x; b < n_bins; b += blockDim.x)
        if (s_sum[b] != 0.0) atomicAdd(&sums[b], s_sum[b]);
}

__global__ void __launch_bounds__(kMaxBins)
k_spectrum_finish(int n_bins, double *__restrict__ sums, const double *__restrict__ dlnr, double rho, double V,
                  int n_smooth, double *__restrict__ out)
{
    __shared__ double s_a[kMaxBins], s_b[kMaxBins];
    const int b = threadIdx.x;
    if (b < n_bins) {
        s_a[b] = __ddiv_rn(__ddiv_rn(__dmul_rn(sums[b], rho), V), dlnr[b]);
        sums[b] = 0.0;                                            // ready for the next call
    }
    __syncthreads();
    double *src = s_a, *dst = s_b;
    for (int pass = 0; pass < n_smooth; ++pass) {
        if (b < n_bins) {
            const int lo = max(b - 2, 0), hi = min(b + 2, n_bins - 1);
            double s = 0.0;
            for (int k = lo; k <= hi; ++k) s = __dadd_rn(s, src[k]);
            dst[b] = __ddiv_rn(s, (double)(hi - lo + 1));
        }
        __syncthreads();
        double *t = src; src = dst; dst = t;
    }
    if (b < n_bins) out[b] = src[b];
}

}  // namespace sdmk
