// K2 -- fused exchange + Coulomb-trace kernel (one launch per spin).
//   T^{w,gamma}_ij = sum_p Ltilde^gamma_ip theta^w_jp      PAPER.md:239 (Eq. 29) -- "the computational bottleneck"
//   x^w   += sum_ij T_ij T_ji                              PAPER.md:234 (Eq. 28), Listing 4
//   t^{w,gamma} = sum_i T_ii                               Coulomb / force-bias trace, PAPER.md:195 (Eq. 24)
// T is formed and consumed on chip ("direct algorithm"): accumulators live in registers, the CTA
// tile passes once through shared memory for the transpose pairing T_ij T_ji, nothing of size Nw*Ngamma*n^2 is
// ever written to global memory.
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
    int LD;                        // leading dimension (doubles) of the staging buffer: 8*NT + 1 (odd)
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
    const int npairs = n * (n + 1) / 2, upb = (npairs + 31) >> 5;                              // pairs i<=j; 32-pair units per block
    int2 *pairtab = reinterpret_cast<int2 *>(staging + (size_t)P.strips * 8 * LD);             // [npairs] (i*LD+j, j*LD+i)
    double *red = reinterpret_cast<double *>(pairtab + npairs);                                 // [K2_MAX_WT][K2_MAX_WM][2]
    uint64_t *full_bar = reinterpret_cast<uint64_t *>(red + K2_MAX_WT * K2_MAX_WM * 2);
    uint64_t *empty_bar = full_bar + P.nstages;

    // pair table: k -> (i, j), i <= j, row-major over the upper triangle
    for (int i = tid; i < n; i += blockDim.x) {
        int k = i * n - (i * (i - 1)) / 2;
        for (int j = i; j < n; ++j, ++k) pairtab[k] = make_int2(i * LD + j, j * LD + i);
    }
    if (tid == 0) {
        for (int s = 0; s < P.nstages; ++s) {
            mbar_init(&full_bar[s], 1);
            mbar_init(&empty_bar[s], WM);
        }
        mbar_fence_init();
    }
    __syncthreads();

    const int last_ks = P.ksteps - (P.nchunks - 1) * P.ksc;
    // Tiles are dealt round-robin, tile index t = rt * n_ct + ct; a CTA steps from t to t + gridDim.x with two adds
    // and a compare (no division on the per-chunk path).
    const int step_rt = (int)(gridDim.x / (unsigned)P.n_ct), step_ct = (int)(gridDim.x % (unsigned)P.n_ct);
    const int first_rt = (int)(blockIdx.x / (unsigned)P.n_ct), first_ct = (int)(blockIdx.x % (unsigned)P.n_ct);

    // ---- producer: lane 0 of the LAST warp (the warp with the fewest strips, i.e. the most slack).  It runs
    // `nstages - 2` chunks ahead of the consumers, so the stage it refills was released by every warp at least one
    // chunk ago and its wait on the empty barrier does not stall.
    const bool is_producer = (tid == (WM - 1) * 32);
    int p_rt = first_rt, p_ct = first_ct, p_chunk = 0, p_stage = 0;
    uint32_t p_phase = 0;
    const double *p_a = P.A + (long long)p_rt * P.tileA_doubles;
    const double *p_b = P.B + (long long)p_ct * P.tileB_doubles;
    auto produce_one = [&]() {
        if (p_rt >= P.n_rt) return;
        const bool last = (p_chunk == P.nchunks - 1);
        const uint32_t ab = last ? (uint32_t)last_ks * P.strips * 256u : a_chunk_bytes;
        const uint32_t bb = last ? (uint32_t)last_ks * NT * 256u : b_chunk_bytes;
        mbar_wait(&empty_bar[p_stage], p_phase ^ 1u);
        mbar_arrive_expect_tx(&full_bar[p_stage], ab + bb);
        unsigned char *dst = stage_base + (size_t)p_stage * stage_bytes;
        bulk_g2s(dst, p_a, ab, &full_bar[p_stage]);
        bulk_g2s(dst + a_chunk_bytes, p_b, bb, &full_bar[p_stage]);
        p_a += a_chunk_bytes / 8; p_b += b_chunk_bytes / 8;
        if (++p_stage == P.nstages) { p_stage = 0; p_phase ^= 1u; }
        if (last) {
            p_chunk = 0;
            p_rt += step_rt; p_ct += step_ct;
            if (p_ct >= P.n_ct) { p_ct -= P.n_ct; ++p_rt; }
            p_a = P.A + (long long)p_rt * P.tileA_doubles;
            p_b = P.B + (long long)p_ct * P.tileB_doubles;
        } else {
            ++p_chunk;
        }
    };
    if (is_producer)
        for (int d = 0; d < P.nstages - 2; ++d) produce_one();

    // ---- consumers: all WM warps ----
    int my_mt = 0;
#pragma unroll
    for (int m = 0; m < MT; ++m)
        if (warp + m * WM < P.strips) my_mt = m + 1;

    int stage = 0;
    uint32_t phase = 0;
    for (int rt = first_rt, ct = first_ct; rt < P.n_rt;) {
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
        // Phase 1: every warp parks its accumulators in the whole-tile staging buffer, staging[row][col] with the
        // tile's own row/column numbering (row = g*n + i, col = (plane*wT + wl)*n + j), leading dimension LD odd.
        const int g0 = rt * P.gT;
        const int gvalid = min(P.gT, P.n_gamma - g0);
        const int w0 = ct * P.wT;
        const int wvalid = min(P.wT, P.n_walkers - w0);
        // (the previous tile's readers all passed its closing barrier, so the buffer is free)
#pragma unroll
        for (int m = 0; m < MT; ++m) {
            if (m < my_mt) {
                double *dst = staging + ((warp + m * WM) * 8 + (lane >> 2)) * LD + 2 * (lane & 3);
#pragma unroll
                for (int q = 0; q < NT; ++q) { dst[q * 8] = acc[m][q][0]; dst[q * 8 + 1] = acc[m][q][1]; }
            }
        }
        named_bar_sync(1, nthr_c);                                         // staging full
        // Phase 2: for every (walker wl, gamma g) block, x += sum_ij T_ij T_ji over the pair table (i <= j, weight 2
        // off the diagonal) and t = sum_i T_ii.  Work unit = 32 consecutive pairs of one block; units are dealt to warps.
        const int planeoff = P.wT * n;
        for (int wl = 0; wl < wvalid; ++wl) {
            double xr = 0.0, xi = 0.0;
            for (int u = warp; u < gvalid * upb; u += WM) {
                const int g = u / upb, kc = u - g * upb;
                const double *Tre = staging + (g * n) * LD + wl * n;
                const double *Tim = Tre + planeoff;
                const int k = kc * 32 + lane;
                if (k < npairs) {
                    const int2 dm = pairtab[k];
                    const double ar = Tre[dm.x], ai = Tim[dm.x], br = Tre[dm.y], bi = Tim[dm.y];
                    const double wgt = (dm.x == dm.y) ? 1.0 : 2.0;
                    double pr = ar * br; pr = fma(-ai, bi, pr);
                    double pi = ar * bi; pi = fma(ai, br, pi);
                    xr = fma(wgt, pr, xr);
                    xi = fma(wgt, pi, xi);
                }
                if (kc == 0) {                                             // uniform per warp: trace of this block
                    double tr = 0.0, ti = 0.0;
                    for (int i = lane; i < n; i += 32) { tr += Tre[i * LD + i]; ti += Tim[i * LD + i]; }
                    tr = warp_sum(tr);
                    ti = warp_sum(ti);
                    if (lane == 0) {
                        double *tp = P.tbuf + ((long long)(w0 + wl) * P.n_gamma + g0 + g) * 2;
                        tp[0] = tr; tp[1] = ti;
                    }
                }
            }
            xr = warp_sum(xr);
            xi = warp_sum(xi);
            if (lane == 0) { red[(wl * K2_MAX_WM + warp) * 2] = xr; red[(wl * K2_MAX_WM + warp) * 2 + 1] = xi; }
        }
        named_bar_sync(2, nthr_c);                                         // red[] complete
        if (tid < wvalid) {
            double sr = 0.0, si = 0.0;
            for (int q = 0; q < WM; ++q) { sr += red[(tid * K2_MAX_WM + q) * 2]; si += red[(tid * K2_MAX_WM + q) * 2 + 1]; }
            double *xp = P.xpart + ((long long)rt * P.maxw + w0 + tid) * 2;
            xp[0] = sr; xp[1] = si;
        }
        rt += step_rt; ct += step_ct;
        if (ct >= P.n_ct) { ct -= P.n_ct; ++rt; }
    }
}

}  // namespace afqmc
