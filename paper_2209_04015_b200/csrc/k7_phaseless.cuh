// K7 -- phaseless weight update (Eq. 7, 8, 10-12), one CTA per walker:
//   O = exp(log_ovlp_new - log_ovlp_old)                          overlap ratio, Eq. 8
//   I = O exp(x . xbar - xbar . xbar / 2)                         importance function, Eq. 7
//   w_new = |I| max(0, cos(arg O)) w                              Eq. 10-12
// x real [Nw][Ngamma] (the sampled auxiliary fields), xbar complex [Nw][Ngamma] (force bias, Eq. 9).  Fixed-order sums.
#pragma once
#include <math_constants.h>
#include "common.cuh"

namespace afqmc {

constexpr int K7_THREADS = 256;

__global__ void __launch_bounds__(K7_THREADS) k7_phaseless_update(int n_gamma, const double *__restrict__ x,
                                                                  const double *__restrict__ xbar,        // [Nw][Ngamma][2]
                                                                  const double *__restrict__ lo_old,      // [Nw][2]
                                                                  const double *__restrict__ lo_new,      // [Nw][2]
                                                                  const double *__restrict__ w_in, double *__restrict__ w_out) {
    const int w = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    __shared__ double s_red[K7_THREADS / 32];
    // only the real part of the exponent enters |I|:  Re(x . xbar) - Re(xbar . xbar) / 2
    double acc = 0.0;
    for (int g = tid; g < n_gamma; g += K7_THREADS) {
        const double xr = xbar[((long long)w * n_gamma + g) * 2], xi = xbar[((long long)w * n_gamma + g) * 2 + 1];
        const double xv = x[(long long)w * n_gamma + g];
        acc = fma(xv, xr, acc);
        acc = fma(-0.5, xr * xr - xi * xi, acc);
    }
    acc = warp_sum(acc);
    if (lane == 0) s_red[warp] = acc;
    __syncthreads();
    if (tid == 0) {
        double e = 0.0;
        for (int q = 0; q < K7_THREADS / 32; ++q) e += s_red[q];
        const double dlog = lo_new[2 * w] - lo_old[2 * w], dphi = lo_new[2 * w + 1] - lo_old[2 * w + 1];
        const double c = cos(dphi);                       // cos(arg O): periodic, no wrapping needed
        w_out[w] = c > 0.0 ? exp(dlog + e) * c * w_in[w] : 0.0;
    }
}

}  // namespace afqmc
