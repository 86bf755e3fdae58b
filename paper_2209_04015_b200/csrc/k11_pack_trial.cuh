// K11 -- packs one spin block of the trial (complex128 [N][n]) into the two operand planes K1's overlap
// product S = psi^dagger phi (Eq. 16) reads: Re psi^T and Im psi^T as DMMA A fragments,
//     plane[((p >> 2) * ns8 + (i >> 3)) * 32 + (i & 7) * 4 + (p & 3)] = Re / Im psi[p][i],     ns8 = ceil(n / 8),
// zero-padded to whole chunks of K1_ROWS rows (the caller clears the planes first).  afqmc_create does this packing on
// the host; the allocation-free entry point afqmc_log_overlap_static does it here, into its static scratch.
#pragma once
#include "common.cuh"

namespace afqmc {

__global__ void __launch_bounds__(256) k11_pack_trial(const double2 *__restrict__ psi, int N, int n, double *__restrict__ plane_re,
                                                      double *__restrict__ plane_im) {
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= N * n) return;
    const int p = idx / n, i = idx - p * n, ns8 = (n + 7) >> 3;
    const long long o = ((long long)(p >> 2) * ns8 + (i >> 3)) * 32 + (i & 7) * 4 + (p & 3);
    const double2 v = psi[idx];
    plane_re[o] = v.x;
    plane_im[o] = v.y;
}

}  // namespace afqmc
