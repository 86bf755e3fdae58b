// K0 -- one-time half-rotation (Eq. 21), executed by afqmc_create, not on the timed path.
//   htilde_sigma[i][p]       = sum_q conj(psi[q][i]) h[q][p]
//   Ltilde^gamma_sigma[i][r] = sum_p conj(psi[p][i]) L^gamma[p][r]      (real trial => real Ltilde)
// Ltilde is written straight into K2's packed A-operand layout (common.cuh).  Both kernels work on one real plane of
// psi at a time (`scale` = +1 for Re psi, -1 for Im psi because of the conjugate); for a complex trial the imaginary
// plane of Ltilde occupies rows n..2n-1 of every gamma block (`row_shift` = n, `rows_per_gamma` = 2n).
#pragma once
#include "common.cuh"

namespace afqmc {

// htilde: one thread per (i, p).
__global__ void k0_half_rotate_h(const double *__restrict__ h1e, const double *__restrict__ psi,  // psi plane [N][n]
                                 int N, int n, double scale, double *__restrict__ ht /* [n][N] */) {
    int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n * N) return;
    int i = idx / N, p = idx - i * N;
    double acc = 0.0;
    for (int q = 0; q < N; ++q) acc = fma(psi[(size_t)q * n + i], h1e[(size_t)q * N + p], acc);
    ht[idx] = scale * acc;
}

// Ltilde: grid = (n_gamma, ceil(N/128)); thread owns one (gamma, r) and produces all i in blocks of 8.
// psi is staged in shared memory by (p-chunk, 8 columns).
constexpr int K0_PCHUNK = 64;

__global__ void __launch_bounds__(128)
k0_half_rotate_chol(const double *__restrict__ chol, const double *__restrict__ psi, int N, int n, int n_gamma,
                    int rows_per_gamma, int row_shift, double scale, OperandLayout lay, double *__restrict__ packedA,
                    OperandLayout layF, double *__restrict__ packedF) {
    // packedA (may be null): K2's exchange operand, rows (gamma, [part,] i), k = p.
    // packedF (may be null): the force-bias operand, rows (gamma[, part]), k = i * N + p   (Eq. 24).
    const int nbf = rows_per_gamma / n, part = row_shift / n;
    __shared__ double psi_s[K0_PCHUNK * 8];  // [K0_PCHUNK][8]
    const int g = blockIdx.x;                                  // gamma on grid.x: no 65535 limit
    const int r = blockIdx.y * blockDim.x + threadIdx.x;
    const double *Lg = chol + (size_t)g * N * N;
    const int tile = packedA ? g / lay.per_tile : 0;           // `lay` is empty when only packedF is wanted
    const int row0 = packedA ? (g - tile * lay.per_tile) * rows_per_gamma + row_shift : 0;
    for (int i0 = 0; i0 < n; i0 += 8) {
        double acc[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) acc[k] = 0.0;
        for (int p0 = 0; p0 < N; p0 += K0_PCHUNK) {
            int pc = min(K0_PCHUNK, N - p0);
            __syncthreads();
            for (int t = threadIdx.x; t < pc * 8; t += blockDim.x) {
                int pp = t >> 3, k = t & 7;
                psi_s[t] = (i0 + k < n) ? psi[(size_t)(p0 + pp) * n + i0 + k] : 0.0;
            }
            __syncthreads();
            if (r < N) {
                for (int pp = 0; pp < pc; ++pp) {
                    double l = Lg[(size_t)(p0 + pp) * N + r];
#pragma unroll
                    for (int k = 0; k < 8; ++k) acc[k] = fma(psi_s[pp * 8 + k], l, acc[k]);
                }
            }
        }
        if (r < N) {
#pragma unroll
            for (int k = 0; k < 8; ++k)
                if (i0 + k < n) {
                    if (packedA) packedA[packed_offset(lay, tile, row0 + i0 + k, r)] = scale * acc[k];
                    if (packedF) {
                        const int tf = g / layF.per_tile;
                        packedF[packed_offset(layF, tf, (g - tf * layF.per_tile) * nbf + part, (i0 + k) * N + r)] = scale * acc[k];
                    }
                }
        }
    }
}

}  // namespace afqmc
