// K1 -- per (walker, spin): overlap matrix, LU with partial pivoting, log-determinant, inverse, theta, E1.
//   S      = psi^dagger phi                 (n x n)                          PAPER.md:143 (Eq. 16), Listing 2 line 1
//   P S    = L U, log det S                                                   PAPER.md:146-150 ("linalg.det"), Listing 2 line 2
//   X      = S^-1
//   theta  = (phi X)^T  (n x N), written as separate re / im planes           PAPER.md:191 (Eq. 23), Listing 2 line 3;
//            in K2's packed B-operand layout (common.cuh)                     re/im split: PAPER.md:260-262, 280
//   E1     = sum_jp htilde_jp theta_jp                                        PAPER.md:282 with Eq. 2, 22
// One CTA per (walker, spin); S and X live in shared memory for the whole kernel.
#pragma once
#include <math_constants.h>
#include "common.cuh"

namespace afqmc {

constexpr int K1_THREADS = 256;
constexpr int K1_PCHUNK = 32;  // rows of phi staged per pass = 8 DMMA k-steps of theta
constexpr int K1_TU = 4;        // DMMA output tiles per warp and pass

struct K1Params {
    const double2 *walkers;       // alpha block [Nw][N][na], then beta block [Nw][N][nb]
    int n_walkers, N, maxw;
    int n[2];
    long long spin_off[2];        // offset of each spin block in `walkers`, in complex elements
    const double *psi[2];         // [N][n] Re psi
    const double *ht[2];          // [n][N] Re htilde
    const double *psi_im[2];      // Im psi, or nullptr for a real trial block
    const double *ht_im[2];       // Im htilde, or nullptr
    double *thetaB[2];            // packed B operand
    OperandLayout layB[2];
    double *thetaF[2];            // force-bias B operand (k = j * N + p, column = plane * wT + wl), or nullptr
    OperandLayout layF[2];
    double *logdet;               // [2][maxw][2]  (log|det|, arg)
    double *e1;                   // [2][maxw][2]
};

__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

template <bool WITH_FB>
__global__ void __launch_bounds__(K1_THREADS, 4) k1_overlap_inverse_theta(K1Params P) {
    const int w = blockIdx.x, sp = blockIdx.y;
    const int n = P.n[sp], N = P.N;
    if (n == 0) return;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    extern __shared__ __align__(16) unsigned char k1_smem[];
    double2 *S = reinterpret_cast<double2 *>(k1_smem);        // [n][n]
    double2 *X = S + n * n;                                   // [n][n]
    double2 *phis = X + n * n;                                // [K1_PCHUNK][n]
    double *psis = reinterpret_cast<double *>(phis + K1_PCHUNK * n);  // [K1_PCHUNK][n]  Re psi
    double *psii = psis + K1_PCHUNK * n;                              // [K1_PCHUNK][n]  Im psi (complex trial)
    int *perm = reinterpret_cast<int *>(psii + K1_PCHUNK * n);        // [n]
    __shared__ int s_piv;
    __shared__ double s_red[2 * (K1_THREADS / 32)];

    const double2 *phi = P.walkers + P.spin_off[sp] + (long long)w * N * n;   // [N][n]
    const double *psi = P.psi[sp];
    const double *psi_im = P.psi_im[sp];
    const bool cplx = psi_im != nullptr;

    // ---- S = psi^dagger phi = (Re psi - i Im psi)^T phi  on the FP64 tensor cores ------------------------------------------
    // Real TN product: rows i (8-row strips), columns (j, re/im) of the interleaved phi (8-column blocks), k = p.
    // Warp `warp` owns the output tiles t = warp + 8 u; a tile's C fragment is exactly S[i][j] as (re, im) per lane.
    const int ns = (n + 7) >> 3, ncb = (2 * n + 7) >> 3, ntile_s = ns * ncb;
    // (K1_TU tiles per warp and pass; n <= 32 needs one pass, larger n re-streams phi once per pass)
    for (int ubase = 0; ubase * 8 < ntile_s; ubase += K1_TU) {
        double sacc[K1_TU][2];
#pragma unroll
        for (int u = 0; u < K1_TU; ++u) { sacc[u][0] = 0.0; sacc[u][1] = 0.0; }
        const int fr = lane >> 2, fk = lane & 3;
        const double *phid = reinterpret_cast<const double *>(phis);
        for (int p0 = 0; p0 < N; p0 += K1_PCHUNK) {
            const int pc = min(K1_PCHUNK, N - p0);
            __syncthreads();
            for (int t = tid; t < pc * n; t += K1_THREADS) {
                phis[t] = phi[(long long)p0 * n + t];
                psis[t] = psi[(long long)p0 * n + t];
                if (cplx) psii[t] = psi_im[(long long)p0 * n + t];
            }
            __syncthreads();
#pragma unroll
            for (int u = 0; u < K1_TU; ++u) {
                const int t = warp + 8 * (ubase + u);
                if (t < ntile_s) {
                    const int st = t / ncb, cb = t - st * ncb;
                    const int i = 8 * st + fr, col = 8 * cb + fr;               // A row / B column of this lane
                    const bool iok = i < n, cok = col < 2 * n;
                    for (int k0 = 0; k0 < pc; k0 += 4) {
                        const int pp = k0 + fk;
                        const bool pok = pp < pc;
                        const double av = (iok && pok) ? psis[pp * n + i] : 0.0;
                        const double bv = (cok && pok) ? phid[pp * 2 * n + col] : 0.0;
                        dmma_m8n8k4(sacc[u][0], sacc[u][1], av, bv);
                        if (cplx) {     // + Im psi^T (phi_im, -phi_re): (a - ib)(x + iy) = (ax + by) + i(ay - bx)
                            const double av2 = (iok && pok) ? psii[pp * n + i] : 0.0;
                            const double sw = (cok && pok) ? phid[pp * 2 * n + (col ^ 1)] : 0.0;
                            dmma_m8n8k4(sacc[u][0], sacc[u][1], av2, (col & 1) ? -sw : sw);
                        }
                    }
                }
            }
        }
#pragma unroll
        for (int u = 0; u < K1_TU; ++u) {
            const int t = warp + 8 * (ubase + u);
            if (t < ntile_s) {
                const int st = t / ncb, cb = t - st * ncb;
                const int i = 8 * st + fr, j = 4 * cb + fk;                     // C fragment: row lane/4, columns 2 (lane%4) + {0, 1}
                if (i < n && j < n) S[i * n + j] = make_double2(sacc[u][0], sacc[u][1]);
            }
        }
    }
    for (int e = tid; e < n; e += K1_THREADS) perm[e] = e;
    __syncthreads();

    // ---- LU with partial pivoting, in place ---------------------------------------------------------
    double logabs = 0.0, ph_re = 1.0, ph_im = 0.0;   // meaningful on thread 0
    bool singular = false;
    for (int k = 0; k < n; ++k) {
        if (warp == 0) {
            double best = -1.0;
            int bi = k;
            for (int i = k + lane; i < n; i += 32) {
                const double2 a = S[i * n + k];
                const double m = a.x * a.x + a.y * a.y;
                if (m > best) { best = m; bi = i; }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const double m2 = __shfl_xor_sync(0xffffffffu, best, o);
                const int i2 = __shfl_xor_sync(0xffffffffu, bi, o);
                if (m2 > best || (m2 == best && i2 < bi)) { best = m2; bi = i2; }
            }
            if (lane == 0) s_piv = bi;
        }
        __syncthreads();
        const int piv = s_piv;
        if (piv != k) {
            for (int j = tid; j < n; j += K1_THREADS) {
                const double2 t = S[k * n + j];
                S[k * n + j] = S[piv * n + j];
                S[piv * n + j] = t;
            }
            if (tid == 0) {
                const int t = perm[k]; perm[k] = perm[piv]; perm[piv] = t;
                ph_re = -ph_re; ph_im = -ph_im;
            }
            __syncthreads();
        }
        const double2 u = S[k * n + k];
        const double m2 = u.x * u.x + u.y * u.y;
        if (m2 == 0.0) { singular = true; break; }      // uniform: every thread reads the same u
        const double2 inv = make_double2(u.x / m2, -u.y / m2);
        if (tid == 0) {
            const double au = sqrt(m2);
            logabs += log(au);
            const double2 ph = cmul(make_double2(ph_re, ph_im), make_double2(u.x / au, u.y / au));
            ph_re = ph.x; ph_im = ph.y;
        }
        for (int i = k + 1 + tid; i < n; i += K1_THREADS) S[i * n + k] = cmul(S[i * n + k], inv);
        __syncthreads();
        const int m = n - k - 1;
        for (int e = tid; e < m * m; e += K1_THREADS) {
            const int ii = e / m;
            const int i = k + 1 + ii, j = k + 1 + (e - ii * m);
            const double2 l = S[i * n + k], r = S[k * n + j];
            double2 a = S[i * n + j];
            a.x -= l.x * r.x - l.y * r.y;
            a.y -= l.x * r.y + l.y * r.x;
            S[i * n + j] = a;
        }
        __syncthreads();
    }

    // ---- X = S^-1 : solve L U X = P -----------------------------------------------------------------
    if (singular) {
        for (int e = tid; e < n * n; e += K1_THREADS) X[e] = make_double2(CUDART_NAN, CUDART_NAN);
        __syncthreads();
    } else {
        for (int e = tid; e < n * n; e += K1_THREADS) {
            const int i = e / n, j = e - i * n;
            X[e] = make_double2(perm[i] == j ? 1.0 : 0.0, 0.0);
        }
        __syncthreads();
        for (int k = 0; k < n - 1; ++k) {                 // forward substitution, unit lower triangle
            const int m = n - k - 1;
            for (int e = tid; e < m * n; e += K1_THREADS) {
                const int ii = e / n;
                const int i = k + 1 + ii, j = e - ii * n;
                const double2 l = S[i * n + k], r = X[k * n + j];
                double2 a = X[i * n + j];
                a.x -= l.x * r.x - l.y * r.y;
                a.y -= l.x * r.y + l.y * r.x;
                X[i * n + j] = a;
            }
            __syncthreads();
        }
        for (int k = n - 1; k >= 0; --k) {                // back substitution, upper triangle
            const double2 u = S[k * n + k];
            const double m2 = u.x * u.x + u.y * u.y;
            const double2 inv = make_double2(u.x / m2, -u.y / m2);
            for (int j = tid; j < n; j += K1_THREADS) X[k * n + j] = cmul(X[k * n + j], inv);
            __syncthreads();
            for (int e = tid; e < k * n; e += K1_THREADS) {
                const int i = e / n, j = e - i * n;
                const double2 l = S[i * n + k], r = X[k * n + j];
                double2 a = X[i * n + j];
                a.x -= l.x * r.x - l.y * r.y;
                a.y -= l.x * r.y + l.y * r.x;
                X[i * n + j] = a;
            }
            __syncthreads();
        }
    }

    // ---- theta_jp = sum_i phi_pi X_ij ; packed write; E1 partial ----------------------------------------
    const OperandLayout lay = P.layB[sp];
    const int wT = lay.per_tile;
    const int tile = w / wT, wl = w - tile * wT;
    const int col_re = wl * n, col_im = (wT + wl) * n;
    double *out = P.thetaB[sp];
    double *outF = WITH_FB ? P.thetaF[sp] : nullptr;
    const OperandLayout layF = P.layF[sp];
    const int tileF = WITH_FB ? w / layF.per_tile : 0, wlF = WITH_FB ? w - tileF * layF.per_tile : 0;
    const double *ht = P.ht[sp];
    const double *ht_im = P.ht_im[sp];
    const int kk = lane & 3, jj = lane >> 2;
    double e1r = 0.0, e1i = 0.0;
    const int Kpad = lay.ksteps * 4;
    for (int p0 = 0; p0 < Kpad; p0 += K1_PCHUNK) {
        const int pc = max(0, min(K1_PCHUNK, N - p0));
        __syncthreads();
        for (int t = tid; t < pc * n; t += K1_THREADS) phis[t] = phi[(long long)p0 * n + t];
        __syncthreads();
        const int pl = warp * 4 + kk;           // 8 warps x 4 = 32 rows of the chunk
        const int p = p0 + pl;
        if (p < Kpad) {
            // two columns j, j + 8 per pass share every phi element fetched (same i order per sum as one column at a time)
            for (int jb = jj; jb < n; jb += 16) {
                double2 acc[2];
#pragma unroll
                for (int t = 0; t < 2; ++t) acc[t] = make_double2(0.0, 0.0);
                const bool j1ok = jb + 8 < n;
                if (p < N) {
                    const double2 *fr = phis + pl * n;
                    const int j1 = j1ok ? jb + 8 : jb;
                    for (int i = 0; i < n; ++i) {
                        const double2 f = fr[i], x0 = X[i * n + jb], x1 = X[i * n + j1];
                        acc[0].x = fma(f.x, x0.x, acc[0].x); acc[0].x = fma(-f.y, x0.y, acc[0].x);
                        acc[0].y = fma(f.x, x0.y, acc[0].y); acc[0].y = fma(f.y, x0.x, acc[0].y);
                        acc[1].x = fma(f.x, x1.x, acc[1].x); acc[1].x = fma(-f.y, x1.y, acc[1].x);
                        acc[1].y = fma(f.x, x1.y, acc[1].y); acc[1].y = fma(f.y, x1.x, acc[1].y);
                    }
                }
#pragma unroll
                for (int t = 0; t < 2; ++t) {
                    const int j = jb + 8 * t;
                    if (t == 1 && !j1ok) continue;
                    if (p < N) {
                        const double hv = ht[(long long)j * N + p];
                        e1r = fma(hv, acc[t].x, e1r);
                        e1i = fma(hv, acc[t].y, e1i);
                        if (cplx) {
                            const double hi = ht_im[(long long)j * N + p];
                            e1r = fma(-hi, acc[t].y, e1r);
                            e1i = fma(hi, acc[t].x, e1i);
                        }
                    }
                    out[packed_offset(lay, tile, col_re + j, p)] = acc[t].x;
                    out[packed_offset(lay, tile, col_im + j, p)] = acc[t].y;
                    if (WITH_FB && p < N) {
                        outF[packed_offset(layF, tileF, wlF, j * N + p)] = acc[t].x;
                        outF[packed_offset(layF, tileF, layF.per_tile + wlF, j * N + p)] = acc[t].y;
                    }
                }
            }
        }
    }

    // ---- deterministic block reduction of E1; outputs ---------------------------------------------------
    e1r = warp_sum(e1r);
    e1i = warp_sum(e1i);
    if (lane == 0) { s_red[2 * warp] = e1r; s_red[2 * warp + 1] = e1i; }
    __syncthreads();
    if (tid == 0) {
        double sr = 0.0, si = 0.0;
        for (int q = 0; q < K1_THREADS / 32; ++q) { sr += s_red[2 * q]; si += s_red[2 * q + 1]; }
        double *e1 = P.e1 + ((long long)sp * P.maxw + w) * 2;
        double *ld = P.logdet + ((long long)sp * P.maxw + w) * 2;
        if (singular) {
            e1[0] = CUDART_NAN; e1[1] = CUDART_NAN;
            ld[0] = -CUDART_INF; ld[1] = 0.0;
        } else {
            e1[0] = sr; e1[1] = si;
            ld[0] = logabs; ld[1] = atan2(ph_im, ph_re);
        }
    }
}

}  // namespace afqmc
