// K3 -- energy assembly, one CTA per walker, fixed reduction order (deterministic).
//   E_w = E0 + E1_w + 1/2 sum_gamma (t^gamma_alpha + t^gamma_beta)^2 - 1/2 sum_sigma sum_tiles xpart
//   log-overlap_w = sum_sigma (log|det S_sigma|, arg det S_sigma), arg wrapped to (-pi, pi]
#pragma once
#include <math_constants.h>
#include "common.cuh"

namespace afqmc {

constexpr int K3_THREADS = 128;

struct K3Params {
    int n_gamma, maxw;
    int n[2];
    int n_rt[2];
    const double *tbuf[2];    // [maxw][n_gamma][2]
    const double *xpart[2];   // [n_rt][maxw][2]
    const double *e1;         // [2][maxw][2]
    const double *logdet;     // [2][maxw][2]
    double e0;
    double *out_energy;       // [Nw][2]
    double *out_overlap;      // [Nw][2]
};

__global__ void __launch_bounds__(K3_THREADS) k3_assemble(K3Params P) {
    const int w = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    __shared__ double s_red[4 * (K3_THREADS / 32)];
    double cr = 0.0, ci = 0.0, xr = 0.0, xi = 0.0;
    for (int g = tid; g < P.n_gamma; g += K3_THREADS) {
        double tr = 0.0, ti = 0.0;
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            if (P.n[s] > 0) {
                const double *t = P.tbuf[s] + ((long long)w * P.n_gamma + g) * 2;
                tr += t[0]; ti += t[1];
            }
        }
        cr += tr * tr - ti * ti;
        ci += 2.0 * tr * ti;
    }
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        if (P.n[s] > 0) {
            for (int r = tid; r < P.n_rt[s]; r += K3_THREADS) {
                const double *x = P.xpart[s] + ((long long)r * P.maxw + w) * 2;
                xr += x[0]; xi += x[1];
            }
        }
    }
    cr = warp_sum(cr); ci = warp_sum(ci); xr = warp_sum(xr); xi = warp_sum(xi);
    if (lane == 0) { s_red[4 * warp] = cr; s_red[4 * warp + 1] = ci; s_red[4 * warp + 2] = xr; s_red[4 * warp + 3] = xi; }
    __syncthreads();
    if (tid == 0) {
        double a = 0.0, b = 0.0, c = 0.0, d = 0.0;
        for (int q = 0; q < K3_THREADS / 32; ++q) { a += s_red[4 * q]; b += s_red[4 * q + 1]; c += s_red[4 * q + 2]; d += s_red[4 * q + 3]; }
        double er = P.e0 + 0.5 * a - 0.5 * c, ei = 0.5 * b - 0.5 * d;
        double la = 0.0, ar = 0.0;
        for (int s = 0; s < 2; ++s) {
            if (P.n[s] > 0) {
                const double *e1 = P.e1 + ((long long)s * P.maxw + w) * 2;
                const double *ld = P.logdet + ((long long)s * P.maxw + w) * 2;
                er += e1[0]; ei += e1[1];
                la += ld[0]; ar += ld[1];
            }
        }
        if (ar > CUDART_PI) ar -= 2.0 * CUDART_PI;
        else if (ar <= -CUDART_PI) ar += 2.0 * CUDART_PI;
        P.out_energy[2 * w] = er; P.out_energy[2 * w + 1] = ei;
        P.out_overlap[2 * w] = la; P.out_overlap[2 * w + 1] = ar;
    }
}

// force bias copy-out: out[w][gamma] = t_alpha + t_beta          PAPER.md:195 (Eq. 24)
__global__ void k3_force_bias(int n_walkers, int n_gamma, int na, int nb, const double *ta, const double *tb, double *out) {
    long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long long)n_walkers * n_gamma * 2) return;
    double v = 0.0;
    if (na > 0) v += ta[idx];
    if (nb > 0) v += tb[idx];
    out[idx] = v;
}

// force bias from the raw products of K2's force-bias mode          PAPER.md:168-170, 195 (Eq. 19, 24)
//   real Ltilde:     xbar = (C[gamma][re w], C[gamma][im w])
//   complex Ltilde:  xbar = (C[re gamma][re w] - C[im gamma][im w],  C[re gamma][im w] + C[im gamma][re w])
struct K4Params {
    int n_walkers, n_gamma;
    int n[2], nb[2], wT[2], n_ct[2], ldc[2];   // nb = rows per gamma (1 or 2), ldc = 8 * NT columns per tile
    int ksplit[2];                              // K parts, summed here in a fixed order
    const double *craw[2];
    double *out;                                // [n_walkers][n_gamma][2]
};

__global__ void k4_force_bias_combine(K4Params P) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long long)P.n_walkers * P.n_gamma) return;
    const int w = (int)(idx / P.n_gamma), g = (int)(idx - (long long)w * P.n_gamma);
    double xr = 0.0, xi = 0.0;
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        if (P.n[s] == 0) continue;
        const int ct = w / P.wT[s], wl = w - ct * P.wT[s];
        const long long part_stride = (long long)P.n_gamma * P.nb[s] * P.n_ct[s] * P.ldc[s];
        for (int k = 0; k < P.ksplit[s]; ++k) {
            const double *c0 = P.craw[s] + k * part_stride + ((long long)(g * P.nb[s]) * P.n_ct[s] + ct) * P.ldc[s];
            xr += c0[wl]; xi += c0[P.wT[s] + wl];
            if (P.nb[s] == 2) {
                const double *c1 = c0 + (long long)P.n_ct[s] * P.ldc[s];
                xr -= c1[P.wT[s] + wl]; xi += c1[wl];
            }
        }
    }
    P.out[2 * idx] = xr; P.out[2 * idx + 1] = xi;
}

}  // namespace afqmc
