// K2 -- fused exchange + Coulomb-trace kernel (one launch per spin).
//   T^{w,gamma}_ij = sum_p Ltilde^gamma_ip theta^w_jp      PAPER.md:239 (Eq. 29) -- "the computational bottleneck"
//   x^w   += sum_ij T_ij T_ji                              PAPER.md:234 (Eq. 28), Listing 4
//   t^{w,gamma} = sum_i T_ii                               Coulomb / force-bias trace, PAPER.md:195 (Eq. 24)
// T is formed and consumed on chip ("direct algorithm"): accumulators live in registers, one
// walker's slice of the CTA tile passes through shared memory for the transpose pairing, nothing of size
// Nw*Ngamma*n^2 is ever written to global memory.
//
// Structure (B200): persistent CTAs, one per SM, WM warps.  Thread 0 doubles as the producer: it issues 1-D bulk
// async copies (TMA engine) of contiguous K-chunks of the packed operands (common.cuh) into a ring of shared-memory
// stages guarded by full/empty mbarriers, nstages-2 chunks ahead of the math (a 13th, dedicated producer warp would
// round the CTA up to 16 warps of register allocation and cap the kernel at 128 registers per thread).
// Every warp is a consumer: each owns up to MT 8-row strips
// (strip s -> warp s % WM) times all NT 8-column blocks of the tile, i.e. up to MT*NT DMMA.8x8x4 accumulators,
// complex arithmetic built from real tiles (real Ltilde x re/im planes of theta).
#pragma once
#include "common.cuh"

namespace afqmc {

constexpr int K2_MAX_WT = 4;       // walkers per CTA tile
constexpr int K2_MAX_WM = 12;      // consumer warps

struct K2Params {
    const double *A;               // packed Ltilde of this spin
    const double *B;               // packed theta planes of this spin
    long long tileA_doubles, tileB_doubles;
    int n, gT, wT;                 // electrons, gamma-blocks per tile, walkers per tile
    int strips;                    // 8-row strips per A tile
    int WM;                        // consumer warps
    int ksteps, ksc, nchunks;      // total k-steps, k-steps per chunk, chunks per tile
    int nstages;
    int n_rt, n_ct;                // row tiles (gamma), column tiles (walkers)
    int n_gamma, n_walkers, maxw;
    int LD;                        // leading dimension (doubles) of the staging buffer, odd
    double *tbuf;                  // [maxw][n_gamma][2]  traces of this spin
    double *xpart;                 // [n_rt][maxw][2]     exchange partial sums of this spin
};

template <int MT, int NT>
__global__ void __maxnreg__(168) k2_exchange(const K2Params P) {   // blockDim <= 32*K2_MAX_WM = 384: 384*168 <= 64K registers
    extern __shared__ __align__(128) unsigned char k2_smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int WM = P.WM, n = P.n, LD = P.LD;
    const int nthr_c = WM * 32;

    const uint32_t a_chunk_bytes = (uint32_t)P.ksc * P.strips * 256u;
    const uint32_t b_chunk_bytes = (uint32_t)P.ksc * NT * 256u;
    const uint32_t stage_bytes = a_chunk_bytes + b_chunk_bytes;
    unsigned char *stage_base = k2_smem;
    double *staging = reinterpret_cast<double *>(k2_smem + (size_t)P.nstages * stage_bytes);   // [8*strips][LD]
    int *colinfo = reinterpret_cast<int *>(staging + (size_t)P.strips * 8 * LD);                // [8*NT]
    double *red = reinterpret_cast<double *>(colinfo + 8 * NT + (8 * NT & 1));                  // [K2_MAX_WT][WM][2]
    uint64_t *full_bar = reinterpret_cast<uint64_t *>(red + K2_MAX_WT * K2_MAX_WM * 2);
    uint64_t *empty_bar = full_bar + P.nstages;

    // column table: c -> (plane, wl, j) packed as plane<<30 | wl<<16 | j ; -1 for padding
    for (int c = tid; c < 8 * NT; c += blockDim.x) {
        int v = -1;
        if (c < 2 * P.wT * n) {
            const int pw = c / n, j = c - pw * n;
            const int plane = pw / P.wT, wl = pw - plane * P.wT;
            v = (plane << 30) | (wl << 16) | j;
        }
        colinfo[c] = v;
    }
    if (tid == 0) {
        for (int s = 0; s < P.nstages; ++s) {
            mbar_init(&full_bar[s], 1);
            mbar_init(&empty_bar[s], WM);
        }
        mbar_fence_init();
    }
    __syncthreads();

    const long long ntiles = (long long)P.n_rt * P.n_ct;
    const int last_ks = P.ksteps - (P.nchunks - 1) * P.ksc;

    // ---- producer cursor (meaningful on warp 0 / lane 0 only): runs `nstages - 2` chunks ahead of the consumers,
    // so the stage it refills was released by every warp at least one chunk ago and the wait never stalls.
    long long p_tile = blockIdx.x;
    int p_chunk = 0, p_stage = 0;
    uint32_t p_phase = 0;
    auto produce_one = [&]() {
        if (p_tile >= ntiles) return;
        const int rt = (int)(p_tile / P.n_ct), ct = (int)(p_tile - (long long)rt * P.n_ct);
        const int nks = (p_chunk == P.nchunks - 1) ? last_ks : P.ksc;
        mbar_wait(&empty_bar[p_stage], p_phase ^ 1u);
        const uint32_t ab = (uint32_t)nks * P.strips * 256u, bb = (uint32_t)nks * NT * 256u;
        mbar_arrive_expect_tx(&full_bar[p_stage], ab + bb);
        unsigned char *dst = stage_base + (size_t)p_stage * stage_bytes;
        bulk_g2s(dst, P.A + (long long)rt * P.tileA_doubles + (long long)p_chunk * P.ksc * P.strips * 32, ab,
                 &full_bar[p_stage]);
        bulk_g2s(dst + a_chunk_bytes, P.B + (long long)ct * P.tileB_doubles + (long long)p_chunk * P.ksc * NT * 32, bb,
                 &full_bar[p_stage]);
        if (++p_stage == P.nstages) { p_stage = 0; p_phase ^= 1u; }
        if (++p_chunk == P.nchunks) { p_chunk = 0; p_tile += gridDim.x; }
    };
    const bool is_producer = (tid == 0);
    if (is_producer)
        for (int d = 0; d < P.nstages - 2; ++d) produce_one();

    // ---- consumers: all WM warps ----
    int my_mt = 0;
#pragma unroll
    for (int m = 0; m < MT; ++m)
        if (warp + m * WM < P.strips) my_mt = m + 1;

    int stage = 0;
    uint32_t phase = 0;
    for (long long t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const int rt = (int)(t / P.n_ct), ct = (int)(t - (long long)rt * P.n_ct);
        double acc[MT][NT][2];
#pragma unroll
        for (int m = 0; m < MT; ++m)
#pragma unroll
            for (int q = 0; q < NT; ++q) { acc[m][q][0] = 0.0; acc[m][q][1] = 0.0; }

        for (int c = 0; c < P.nchunks; ++c) {
            const int nks = (c == P.nchunks - 1) ? last_ks : P.ksc;
            if (is_producer) produce_one();
            __syncwarp();
            mbar_wait(&full_bar[stage], phase);
            const double *As = reinterpret_cast<const double *>(stage_base + (size_t)stage * stage_bytes);
            const double *Bs = reinterpret_cast<const double *>(stage_base + (size_t)stage * stage_bytes + a_chunk_bytes);
            for (int ks = 0; ks < nks; ++ks) {
                double a[MT], b[NT];
#pragma unroll
                for (int m = 0; m < MT; ++m)
                    a[m] = (m < my_mt) ? As[(ks * P.strips + warp + m * WM) * 32 + lane] : 0.0;
#pragma unroll
                for (int q = 0; q < NT; ++q) b[q] = Bs[(ks * NT + q) * 32 + lane];
#pragma unroll
                for (int m = 0; m < MT; ++m) {
                    if (m < my_mt) {
#pragma unroll
                        for (int q = 0; q < NT; ++q) dmma_m8n8k4(acc[m][q][0], acc[m][q][1], a[m], b[q]);
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_bar[stage]);
            if (++stage == P.nstages) { stage = 0; phase ^= 1u; }
        }

        // ------------------------------ epilogue ------------------------------
        const int g0 = rt * P.gT;
        const int gvalid = min(P.gT, P.n_gamma - g0);
        const int rows_valid = gvalid * n;
        for (int wl = 0; wl < P.wT; ++wl) {
            const int w = ct * P.wT + wl;
            if (w >= P.n_walkers) break;                                   // uniform
            named_bar_sync(1, nthr_c);                                     // staging free
#pragma unroll
            for (int m = 0; m < MT; ++m) {
                if (m < my_mt) {
                    const int row = (warp + m * WM) * 8 + (lane >> 2);
#pragma unroll
                    for (int q = 0; q < NT; ++q) {
#pragma unroll
                        for (int e = 0; e < 2; ++e) {
                            const int ci = colinfo[q * 8 + 2 * (lane & 3) + e];
                            if (ci >= 0 && ((ci >> 16) & 0x3fff) == wl) {
                                const int plane = (ci >> 30) & 1, j = ci & 0xffff;
                                staging[row * LD + plane * n + j] = acc[m][q][e];
                            }
                        }
                    }
                }
            }
            named_bar_sync(1, nthr_c);                                     // staging full
            // exchange: sum over (g,i,j) of T_ij T_ji ;  T_ij = staging[g*n+i][j] + i staging[g*n+i][n+j]
            double xr = 0.0, xi = 0.0;
            for (int item = tid; item < 2 * rows_valid; item += nthr_c) {
                const int half = item >= rows_valid;
                const int r = item - half * rows_valid;
                const int g = r / n, i = r - g * n;
                const double *rowp = staging + r * LD;
                const double *mir = staging + (g * n) * LD + i;
                for (int j = half; j < n; j += 2) {
                    const double ar = rowp[j], ai = rowp[n + j];
                    const double br = mir[j * LD], bi = mir[j * LD + n];
                    xr = fma(ar, br, xr); xr = fma(-ai, bi, xr);
                    xi = fma(ar, bi, xi); xi = fma(ai, br, xi);
                }
            }
            // traces
            if (tid < gvalid) {
                double tr = 0.0, ti = 0.0;
                const double *d = staging + (tid * n) * LD;
                for (int i = 0; i < n; ++i) { tr += d[i * LD + i]; ti += d[i * LD + n + i]; }
                double *tp = P.tbuf + ((long long)w * P.n_gamma + g0 + tid) * 2;
                tp[0] = tr; tp[1] = ti;
            }
            xr = warp_sum(xr);
            xi = warp_sum(xi);
            if (lane == 0) { red[(wl * K2_MAX_WM + warp) * 2] = xr; red[(wl * K2_MAX_WM + warp) * 2 + 1] = xi; }
        }
        named_bar_sync(1, nthr_c);
        if (tid < P.wT) {
            const int w = ct * P.wT + tid;
            if (w < P.n_walkers) {
                double sr = 0.0, si = 0.0;
                for (int q = 0; q < WM; ++q) { sr += red[(tid * K2_MAX_WM + q) * 2]; si += red[(tid * K2_MAX_WM + q) * 2 + 1]; }
                double *xp = P.xpart + ((long long)rt * P.maxw + w) * 2;
                xp[0] = sr; xp[1] = si;
            }
        }
    }
}

}  // namespace afqmc
