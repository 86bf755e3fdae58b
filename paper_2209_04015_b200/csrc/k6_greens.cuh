// K6 -- optional full one-body Green's function of one spin sector (the paper's `greens_function(..., build_full=True)`,
// PAPER.md:412-414, for user-written mixed estimators such as Listing 6):
//   G^sigma_pq = [phi (psi^dagger phi)^-1 psi^dagger]_qp = sum_j theta^sigma_jq conj(psi^sigma_pj)     PAPER.md:187 (Eq. 22, the
//   matrix form; its last member, sum_j theta_jp (psi^dagger)_jq, is the transpose of it -- DESIGN.md section 3 #16)
// from the theta planes K1 left in the handle (packed B operand, common.cuh).  Output [Nw][N][N] complex128, row-major
// in (p, q).  Grid (Nw, ceil(N/32), ceil(N/32)), 256 threads: a 32 x 32 tile of G per CTA, 4 elements per thread.
#pragma once
#include "common.cuh"

namespace afqmc {

constexpr int K6_TILE = 32;

struct K6Params {
    int N, n;
    const double *theta;            // packed B operand of this spin
    OperandLayout layB;
    const double *psi, *psi_im;     // [N][n] planes, psi_im may be nullptr
    double2 *out;                   // [Nw][N][N]
};

__global__ void __launch_bounds__(256) k6_greens_function(K6Params P) {
    extern __shared__ __align__(16) unsigned char k6_smem[];
    const int n = P.n, N = P.N, w = blockIdx.x;               // walker on grid.x: no 65535 limit
    const int p0 = blockIdx.y * K6_TILE, q0 = blockIdx.z * K6_TILE;
    double2 *th = reinterpret_cast<double2 *>(k6_smem);       // [n][32]  theta_jq for the tile's q
    double2 *ps = th + n * K6_TILE;                           // [n][32]  conj(psi_pj) for the tile's p
    const OperandLayout lay = P.layB;
    const int tile = w / lay.per_tile, wl = w - tile * lay.per_tile;
    for (int t = threadIdx.x; t < n * K6_TILE; t += 256) {
        const int j = t / K6_TILE, pp = t - j * K6_TILE;
        const int p = p0 + pp, q = q0 + pp;
        th[t] = q < N ? make_double2(P.theta[packed_offset(lay, tile, wl * n + j, q)],
                                     P.theta[packed_offset(lay, tile, (lay.per_tile + wl) * n + j, q)])
                      : make_double2(0.0, 0.0);
        ps[t] = p < N ? make_double2(P.psi[(long long)p * n + j], P.psi_im ? -P.psi_im[(long long)p * n + j] : 0.0)
                      : make_double2(0.0, 0.0);
    }
    __syncthreads();
    const int qq = threadIdx.x & 31, pb = threadIdx.x >> 5;    // q fastest: coalesced stores
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int pp = pb + 8 * r;
        double gr = 0.0, gi = 0.0;
        for (int j = 0; j < n; ++j) {
            const double2 a = ps[j * K6_TILE + pp], b = th[j * K6_TILE + qq];
            gr = fma(a.x, b.x, gr); gr = fma(-a.y, b.y, gr);
            gi = fma(a.x, b.y, gi); gi = fma(a.y, b.x, gi);
        }
        if (p0 + pp < N && q0 + qq < N) P.out[((long long)w * N + p0 + pp) * N + q0 + qq] = make_double2(gr, gi);
    }
}

}  // namespace afqmc
