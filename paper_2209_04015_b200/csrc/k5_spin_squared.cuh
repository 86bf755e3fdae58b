// K5 -- <S^2> mixed estimator for a single-determinant trial (Eq. 31; Listing 6):
//   s2_w = N_dn + M_S (M_S + 1) - sum_pq G^up_pq G^dn_qp ,      M_S = (n_up - n_dn) / 2,
// evaluated in half-rotated form (no N x N Green's function is built):  with G^s_pq = sum_j theta^s_jq conj(psi^s_pj)
// (Eq. 22, matrix form)
//   sum_pq G^up_pq G^dn_qp = sum_jk A_jk B_kj ,   A = theta^up conj(psi^dn)  (n_up x n_dn),   B = theta^dn conj(psi^up)  (n_dn x n_up).
// theta is read from the packed planes K1 wrote for K2 (common.cuh).  One CTA per walker, fixed-order reduction.
#pragma once
#include "common.cuh"

namespace afqmc {

constexpr int K5_THREADS = 256;
constexpr int K5_PCHUNK = 16;

struct K5Params {
    int N, n_walkers;
    int n[2];                       // n_up (alpha), n_dn (beta)
    const double *theta[2];         // packed B operands of K2
    OperandLayout layB[2];
    const double *psi[2];           // [N][n] Re psi
    const double *psi_im[2];        // Im psi or nullptr
    double *out;                    // [n_walkers][2]
};

__global__ void __launch_bounds__(K5_THREADS) k5_spin_squared(K5Params P) {
    const int w = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int na = P.n[0], nb = P.n[1], N = P.N;
    const double ms = 0.5 * (na - nb);
    __shared__ double s_red[2 * (K5_THREADS / 32)];
    if (na == 0 || nb == 0) {
        if (tid == 0) { P.out[2 * w] = nb + ms * (ms + 1.0); P.out[2 * w + 1] = 0.0; }
        return;
    }
    extern __shared__ __align__(16) unsigned char k5_smem[];
    double2 *A = reinterpret_cast<double2 *>(k5_smem);          // [na][nb]
    double2 *B = A + na * nb;                                   // [nb][na]
    double2 *th[2], *ps[2];
    th[0] = B + na * nb;                                        // theta^up chunk [na][PCHUNK]
    th[1] = th[0] + na * K5_PCHUNK;                             // theta^dn chunk [nb][PCHUNK]
    ps[0] = th[1] + nb * K5_PCHUNK;                             // conj(psi^up) chunk [PCHUNK][na]
    ps[1] = ps[0] + na * K5_PCHUNK;                             // conj(psi^dn) chunk [PCHUNK][nb]
    for (int e = tid; e < na * nb; e += K5_THREADS) { A[e] = make_double2(0.0, 0.0); B[e] = make_double2(0.0, 0.0); }
    for (int p0 = 0; p0 < N; p0 += K5_PCHUNK) {
        const int pc = min(K5_PCHUNK, N - p0);
        __syncthreads();
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            const int n = P.n[s];
            const OperandLayout lay = P.layB[s];
            const int tile = w / lay.per_tile, wl = w - tile * lay.per_tile;
            for (int t = tid; t < n * pc; t += K5_THREADS) {
                const int j = t / pc, pp = t - j * pc;
                th[s][j * K5_PCHUNK + pp] = make_double2(P.theta[s][packed_offset(lay, tile, wl * n + j, p0 + pp)],
                                                         P.theta[s][packed_offset(lay, tile, (lay.per_tile + wl) * n + j, p0 + pp)]);
            }
            for (int t = tid; t < pc * n; t += K5_THREADS) {
                const int pp = t / n;
                ps[s][t] = make_double2(P.psi[s][(long long)p0 * n + t], P.psi_im[s] ? -P.psi_im[s][(long long)p0 * n + t] : 0.0);
                (void)pp;
            }
        }
        __syncthreads();
        for (int e = tid; e < na * nb; e += K5_THREADS) {
            const int j = e / nb, k = e - j * nb;                // A_jk += sum_p theta^up_jp conj(psi^dn_pk)
            double2 a = A[e];
            for (int pp = 0; pp < pc; ++pp) {
                const double2 t = th[0][j * K5_PCHUNK + pp], c = ps[1][pp * nb + k];
                a.x = fma(t.x, c.x, a.x); a.x = fma(-t.y, c.y, a.x);
                a.y = fma(t.x, c.y, a.y); a.y = fma(t.y, c.x, a.y);
            }
            A[e] = a;
            const int k2 = e / na, j2 = e - k2 * na;             // B_kj += sum_q theta^dn_kq conj(psi^up_qj)
            double2 b = B[e];
            for (int pp = 0; pp < pc; ++pp) {
                const double2 t = th[1][k2 * K5_PCHUNK + pp], c = ps[0][pp * na + j2];
                b.x = fma(t.x, c.x, b.x); b.x = fma(-t.y, c.y, b.x);
                b.y = fma(t.x, c.y, b.y); b.y = fma(t.y, c.x, b.y);
            }
            B[e] = b;
        }
    }
    __syncthreads();
    double sr = 0.0, si = 0.0;
    for (int e = tid; e < na * nb; e += K5_THREADS) {
        const int j = e / nb, k = e - j * nb;
        const double2 a = A[e], b = B[k * na + j];
        sr = fma(a.x, b.x, sr); sr = fma(-a.y, b.y, sr);
        si = fma(a.x, b.y, si); si = fma(a.y, b.x, si);
    }
    sr = warp_sum(sr); si = warp_sum(si);
    if (lane == 0) { s_red[2 * warp] = sr; s_red[2 * warp + 1] = si; }
    __syncthreads();
    if (tid == 0) {
        double tr = 0.0, ti = 0.0;
        for (int q = 0; q < K5_THREADS / 32; ++q) { tr += s_red[2 * q]; ti += s_red[2 * q + 1]; }
        P.out[2 * w] = nb + ms * (ms + 1.0) - tr;
        P.out[2 * w + 1] = -ti;
    }
}

}  // namespace afqmc
