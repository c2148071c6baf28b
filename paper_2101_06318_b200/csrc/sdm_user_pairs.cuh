// sdm_user_pairs.cuh -- rows a4-a6 around USER-SUPPLIED kernel code ("potentially user-supplied kernel
// code"; the second kernel family of Fig. 8).
//
// This file is never compiled by nvcc: together with sdm_device.cuh it is embedded in libsdm as text and compiled at run
// time by NVRTC (sm_100a, --fmad=false) in ONE translation unit with the caller's source, which defines
//     __device__ double sdm_user_kernel(double vj, double vk, const double *params);
// (vj: volume of the pair member with the larger multiplicity).  The permutation (rows a1-a3) is produced by the
// library's own kernels with collisions switched off; this kernel then walks the candidate pairs (idx[s+2m], idx[s+2m+1])
// of every cell exactly like the built-in pair code: same Philox uniform, same collide_pair arithmetic, every extensive
// attribute, so a user kernel that re-expresses a built-in one reproduces it bit for bit.
// One thread per sorted position p; the thread of a first-in-pair position evaluates the pair.
extern "C" __global__ void __launch_bounds__(256)
k_user_pairs(long long *__restrict__ xi, double *__restrict__ v, const int *__restrict__ cell, const int *__restrict__ idx,
             const int *__restrict__ cell_start, const int *__restrict__ n_ptr, int *__restrict__ zero_count,
             unsigned long long *__restrict__ n_events, unsigned long long *__restrict__ n_exact,
             const sdmk::StepParams prm)
{
    using namespace sdmk;
    const int n = *n_ptr;
    int events = 0, zeros = 0, exact = 0;
    for (int p = blockIdx.x * blockDim.x + threadIdx.x; p + 1 < n; p += gridDim.x * blockDim.x) {
        const int a = idx[p];
        const int c = cell[a];
        const int cs = cell_start[c], ce = cell_start[c + 1];
        if (((p - cs) & 1) != 0 || p + 1 >= ce) continue;         // second-in-pair, or the odd one out of its cell
        const int b = idx[p + 1];
        const double u = block_uniform(droplet_block((uint32_t)a, prm.step, prm.rk));
        const int r = collide_pair_exact<false>(reinterpret_cast<int64_t *>(xi), v, a, b, u, pair_norm(ce - cs, prm.dtdv),
                                                prm.kernel, prm.kparam, prm.attr);
        events += r & 1;
        zeros += (r >> 1) & 1;
        exact += 1;
    }
    events = __reduce_add_sync(0xffffffffu, events);
    zeros = __reduce_add_sync(0xffffffffu, zeros);
    exact = __reduce_add_sync(0xffffffffu, exact);
    if ((threadIdx.x & 31) == 0) {
        if (events) atomicAdd(n_events, (unsigned long long)events);
        if (zeros) atomicAdd(zero_count, zeros);
        if (exact) atomicAdd(n_exact, (unsigned long long)exact);
    }
}
