// K10 -- auxiliary-field sampler of the propagation step: x[w][gamma] ~ N(0, 1)  (Eq. 4: "p(x) is the normal
// distribution"; one vector of Ngamma fields per walker and step).
// Counter-based, so no state is kept and a walker's fields do not depend on the batch it is in (row 21):
//     key = (seed lo, seed hi),  counter = (pair b = gamma / 2, walker, step lo, step hi)
//     (r0, r1, r2, r3) = Philox4x32-10(counter, key)          Salmon et al., SC'11: ten rounds of two 32 x 32 -> 64 multiplies
//     u1 = (((r1:r0) >> 11) + 0.5) 2^-53,  u2 = (((r3:r2) >> 11) + 0.5) 2^-53        in (0, 1), never 0 or 1
//     x[2b] = sqrt(-2 ln u1) cos(2 pi u2),  x[2b + 1] = sqrt(-2 ln u1) sin(2 pi u2)  Box-Muller
// One thread per pair; the integer stream is bit-exact against any other implementation of the algorithm, the normals
// agree with a libm evaluation to a few ulp.
#pragma once
#include <math_constants.h>
#include "common.cuh"

namespace afqmc {

__device__ __forceinline__ void philox4x32_10(uint32_t &c0, uint32_t &c1, uint32_t &c2, uint32_t &c3, uint32_t k0, uint32_t k1) {
#pragma unroll
    for (int rnd = 0; rnd < 10; ++rnd) {
        if (rnd) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
        const uint32_t h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        const uint32_t h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
        c0 = h1 ^ c1 ^ k0; c1 = l1; c2 = h0 ^ c3 ^ k1; c3 = l0;
    }
}

__global__ void __launch_bounds__(256) k10_sample_fields(unsigned long long seed, unsigned long long step, int first_walker, int n_walkers,
                                                         int n_gamma, double *__restrict__ x) {
    const int nb = (n_gamma + 1) >> 1;
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long long)n_walkers * nb) return;
    const int w = (int)(idx / nb), b = (int)(idx - (long long)w * nb);
    uint32_t c0 = (uint32_t)b, c1 = (uint32_t)(first_walker + w), c2 = (uint32_t)step, c3 = (uint32_t)(step >> 32);
    philox4x32_10(c0, c1, c2, c3, (uint32_t)seed, (uint32_t)(seed >> 32));
    const double u1 = ((double)((((unsigned long long)c1 << 32) | c0) >> 11) + 0.5) * 0x1p-53;
    const double u2 = ((double)((((unsigned long long)c3 << 32) | c2) >> 11) + 0.5) * 0x1p-53;
    const double rad = sqrt(-2.0 * log(u1));
    double s, c;
    sincos(2.0 * CUDART_PI * u2, &s, &c);
    double *row = x + (long long)w * n_gamma;
    row[2 * b] = rad * c;
    if (2 * b + 1 < n_gamma) row[2 * b + 1] = rad * s;
}

}  // namespace afqmc
