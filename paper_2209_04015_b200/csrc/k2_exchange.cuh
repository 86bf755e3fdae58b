// K2 -- fused exchange + Coulomb-trace kernel (one launch per spin).
//   T^{w,gamma}_ij = sum_p Ltilde^gamma_ip theta^w_jp      PAPER.md:239 (Eq. 29) -- "the computational bottleneck"
//   x^w   += sum_ij T_ij T_ji                              PAPER.md:234 (Eq. 28), Listing 4
//   t^{w,gamma} = sum_i T_ii                               Coulomb / force-bias trace, PAPER.md:195 (Eq. 24)
// T is formed and consumed on chip ("direct algorithm"): accumulators live in registers, the CTA
// tile passes once through shared memory for the transpose pairing T_ij T_ji, nothing of size Nw*Ngamma*n^2 is
// ever written to global memory.
//
// Structure (B200): persistent CTAs, one per SM, WM warps, every warp an MMA warp.  Each warp owns up to MT 8-row
// strips (strip s -> warp s % WM, so the load is balanced over the 4 SM sub-partitions) times all NT 8-column blocks
// of the tile, i.e. up to MT*NT DMMA.8x8x4 accumulators; complex arithmetic is built from real tiles (real Ltilde x
// re/im planes of theta).  Lane 0 of the last strip-owning warp doubles as the producer: it issues 1-D
// bulk async copies (TMA engine) of contiguous K-chunks of the packed operands (common.cuh) into a ring of
// shared-memory stages guarded by full/empty mbarriers, and never blocks.  The epilogue hands the tile over through
// two more mbarriers (staging full / staging free) instead of CTA-wide barriers.  DESIGN.md section 6 has the
// measurements behind these choices.
#pragma once
#include <type_traits>
#include "common.cuh"

// Timing ablations (results are WRONG, only the time is meaningful; never define this in a product build; build.py passes
// AFQMC_NVCC_EXTRA through):  -DAFQMC_K2_ABLATE=1  epilogue parks the accumulators but skips phase 2 (the T_ij T_ji sums);
// =2  no epilogue at all (K loop only);  =3  K loop without the ring's full / empty barriers and without the producer
// (the operands are whatever the shared memory holds) and no epilogue.  profiles/r2_k2_ablations.md has the numbers.
#ifndef AFQMC_K2_ABLATE
#define AFQMC_K2_ABLATE 0
#endif

namespace afqmc {

constexpr int K2_MAX_WT = 4;       // walkers per CTA tile
constexpr int K2_MAX_WM = 12;      // consumer warps

struct K2Params {
    const double *A;               // packed Ltilde of this spin
    const double *B;               // packed theta planes of this spin
    long long tileA_doubles, tileB_doubles;
    int n, gT, wT;                 // electrons, gamma-blocks per tile, walkers per tile
    int nb, cplx;                  // rows per gamma block of A: n (real Ltilde) or 2n (rows n..2n-1 = Im Ltilde, cplx = 1)
    int strips;                    // 8-row strips per A tile
    int WM;                        // consumer warps
    int ksteps, ksc, nchunks;      // total k-steps, k-steps per chunk, chunks per tile
    int nstages;
    int n_rt, n_ct;                // row tiles (gamma), column tiles (walkers)
    int n_gamma, n_walkers, maxw;
    int H, LD2;                    // staging buffer: row pair pitch LD2 (= 1 mod 16), odd-row offset H (= 8 mod 16)
    double *tbuf;                  // [maxw][n_gamma][2]  traces of this spin
    double *xpart;                 // [n_rt][maxw][2]     exchange partial sums of this spin
};

// Shared-memory fragment load with a compile-time byte offset.  Loads and DMMAs are both `asm volatile`, so the
// software pipeline below is emitted in exactly the order written.
template <int OFF>
__device__ __forceinline__ double lds_f64(uint32_t addr) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1+%2];\n" : "=d"(v) : "r"(addr), "n"(OFF));
    return v;
}

// Ring position of the consumer side of the operand pipeline (identical in every warp).
struct K2Ring {
    uint32_t smem_base;            // shared-window address of stage 0
    uint32_t stage_bytes, a_chunk_bytes, a_kstride;   // a_kstride = strips * 256
    uint32_t full_bar, empty_bar;  // shared-window addresses of the barrier arrays
    int nstages, ksc, nchunks, last_ks, ksteps;
    int stage;
    uint32_t phase;
};

__device__ __forceinline__ void mbar_wait_addr(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP_A:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra.uni WAIT_DONE_A;\n"
        "bra.uni WAIT_LOOP_A;\n"
        "WAIT_DONE_A:\n"
        "}\n" ::"r"(bar), "r"(parity)
        : "memory");
}

__device__ __forceinline__ bool mbar_test_addr(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}

// Wait for a "full" barrier.  The producer warp keeps refilling released stages while it waits, so that the ring
// cannot run dry behind warps that trail it (the epilogue warps).
template <class Produce>
__device__ __forceinline__ void k2_wait_full(uint32_t bar, uint32_t parity, const bool producer_warp, const int lane, Produce &produce_poll) {
    if (producer_warp) {
        while (!mbar_test_addr(bar, parity))
            if (lane == 0) produce_poll();
        __syncwarp();
    } else {
        mbar_wait_addr(bar, parity);
    }
}

// One output tile of one warp: MM strips x NT column blocks, K loop over all chunks / k-steps of the tile.  Per k-step:
// MM + NT fragment loads (256 contiguous bytes per warp each), then MM * NT DMMAs.  Loads and DMMAs are `asm volatile`
// and the strip count MM is a template parameter, so the loop carries no predication and no reconvergence points.
template <int MM, int NT, class Produce>
__device__ __forceinline__ void k2_tile_mma(double (&acc)[MM][NT][2], K2Ring &R, const uint32_t frag_off, const uint32_t a_moff,
                                            const bool producer_warp, Produce &produce_poll, const int lane) {
#pragma unroll 1
    for (int c = 0; c < R.nchunks; ++c) {
        const int nks = (c == R.nchunks - 1) ? R.last_ks : R.ksc;
#if AFQMC_K2_ABLATE != 3
        if (producer_warp) {                       // refill at most one released stage per chunk, never blocking
            if (lane == 0) produce_poll();
            __syncwarp();
        }
        k2_wait_full(R.full_bar + 8u * R.stage, R.phase, producer_warp, lane, produce_poll);
#endif
        uint32_t pa = R.smem_base + R.stage * R.stage_bytes + frag_off;          // + warp * 256 + lane * 8 (in frag_off)
        uint32_t pb = R.smem_base + R.stage * R.stage_bytes + R.a_chunk_bytes + 8u * lane;
#pragma unroll 1
        for (int ks = 0; ks < nks; ++ks) {
            double a[MM], b[NT];
#pragma unroll
            for (int m = 0; m < MM; ++m) a[m] = lds_f64<0>(pa + m * a_moff);
#pragma unroll
            for (int q = 0; q < NT; ++q) b[q] = lds_f64<0>(pb + q * 256);
#pragma unroll
            for (int m = 0; m < MM; ++m)
#pragma unroll
                for (int q = 0; q < NT; ++q) dmma_m8n8k4(acc[m][q][0], acc[m][q][1], a[m], b[q]);
            pa += R.a_kstride;
            pb += NT * 256u;
        }
#if AFQMC_K2_ABLATE != 3
        __syncwarp();
        if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(R.empty_bar + 8u * R.stage) : "memory");
#endif
        if (++R.stage == R.nstages) { R.stage = 0; R.phase ^= 1u; }
    }
}

template <int MT, int NT>
__global__ void __maxnreg__(168) k2_exchange(const K2Params P) {   // blockDim <= 32*K2_MAX_WM = 384: 384*168 <= 64K registers
    extern __shared__ __align__(128) unsigned char k2_smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int WM = P.WM, n = P.n, H = P.H, LD2 = P.LD2;

    const uint32_t a_chunk_bytes = (uint32_t)P.ksc * P.strips * 256u;
    const uint32_t b_chunk_bytes = (uint32_t)P.ksc * NT * 256u;
    const uint32_t stage_bytes = a_chunk_bytes + b_chunk_bytes;
    unsigned char *stage_base = k2_smem;
    double *staging = reinterpret_cast<double *>(k2_smem + (size_t)P.nstages * stage_bytes);   // [4*strips][LD2]
    double *red = staging + (size_t)P.strips * 4 * LD2;                                         // [2][K2_MAX_WT][K2_MAX_WM][2]
    uint64_t *full_bar = reinterpret_cast<uint64_t *>(red + 2 * K2_MAX_WT * K2_MAX_WM * 2);
    uint64_t *empty_bar = full_bar + P.nstages;
    uint64_t *stg_full = empty_bar + P.nstages;          // every warp has parked its accumulators of this tile
    uint64_t *stg_free = stg_full + 1;                   // every warp is done reading the staging buffer
    const int mma_warps = min(WM, P.strips);             // warps that own at least one strip
    if (tid == 0) {
        for (int s = 0; s < P.nstages; ++s) {
            mbar_init(&full_bar[s], 1);
            mbar_init(&empty_bar[s], mma_warps);
        }
        mbar_init(stg_full, WM);
        mbar_init(stg_free, WM);
        mbar_fence_init();
    }
    __syncthreads();

    const int last_ks = P.ksteps - (P.nchunks - 1) * P.ksc;
    // Tiles are dealt round-robin, tile index t = rt * n_ct + ct; a CTA steps from t to t + gridDim.x with two adds
    // and a compare (no division on the per-chunk path).
    const int step_rt = (int)(gridDim.x / (unsigned)P.n_ct), step_ct = (int)(gridDim.x % (unsigned)P.n_ct);
    const int first_rt = (int)(blockIdx.x / (unsigned)P.n_ct), first_ct = (int)(blockIdx.x % (unsigned)P.n_ct);

    // ---- producer: lane 0 of the last strip-owning warp (an epilogue warp, so it has slack).  It issues 1-D bulk async copies (TMA engine) of whole K-chunks of the packed
    // operands into the ring.  It never blocks: once per k-step (and while it waits for its own data) it tests the
    // empty barrier of the next stage to refill and issues the copies if every strip-owning warp has released it.
    const bool producer_warp = (warp == mma_warps - 1);
    int p_rt = first_rt, p_ct = first_ct, p_chunk = 0, p_stage = 0;
    uint32_t p_phase = 0;
    const double *p_a = P.A + (long long)p_rt * P.tileA_doubles;
    const double *p_b = P.B + (long long)p_ct * P.tileB_doubles;
    auto produce_poll = [&]() {
        if (p_rt >= P.n_rt) return;
        if (!mbar_test_addr(smem_u32(&empty_bar[p_stage]), p_phase ^ 1u)) return;
        const bool last = (p_chunk == P.nchunks - 1);
        const uint32_t ab = last ? (uint32_t)last_ks * P.strips * 256u : a_chunk_bytes;
        const uint32_t bb = last ? (uint32_t)last_ks * NT * 256u : b_chunk_bytes;
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
    if (producer_warp && lane == 0)
        for (int d = 0; d < P.nstages; ++d) produce_poll();     // fresh barriers: fills the whole ring

    // ---- every warp: strips warp, warp + WM, ... (my_mt of them: MT or MT - 1, uniform per warp) ----
    int my_mt = 0;
#pragma unroll
    for (int m = 0; m < MT; ++m)
        if (warp + m * WM < P.strips) my_mt = m + 1;

    K2Ring R;
    R.smem_base = smem_u32(stage_base); R.stage_bytes = stage_bytes; R.a_chunk_bytes = a_chunk_bytes;
    asm volatile("" : "+r"(R.smem_base));      // opaque: keeps the window address in a register (no S2R per chunk)
    R.a_kstride = (uint32_t)P.strips * 256u;
    R.full_bar = smem_u32(full_bar); R.empty_bar = smem_u32(empty_bar);
    asm volatile("" : "+r"(R.full_bar), "+r"(R.empty_bar));
    R.nstages = P.nstages; R.ksc = P.ksc; R.nchunks = P.nchunks; R.last_ks = last_ks; R.ksteps = P.ksteps;
    R.stage = 0; R.phase = 0;
    const uint32_t frag_off = (uint32_t)warp * 256u + 8u * lane, a_moff = (uint32_t)WM * 256u;

    // The tile loop is instantiated for the two possible strip counts so that the K loop carries no predication.
    auto run_tiles = [&](auto mm_tag) {
        constexpr int MM = decltype(mm_tag)::value;
        constexpr int MMA = MM > 0 ? MM : 1;
        uint32_t tpar = 0;                                      // parity of this CTA's tile counter
        for (int rt = first_rt, ct = first_ct; rt < P.n_rt;) {
            double acc[MMA][NT][2];
            if constexpr (MM > 0) {
#pragma unroll
                for (int m = 0; m < MM; ++m)
#pragma unroll
                    for (int q = 0; q < NT; ++q) { acc[m][q][0] = 0.0; acc[m][q][1] = 0.0; }
                k2_tile_mma<MM, NT>(acc, R, frag_off, a_moff, producer_warp, produce_poll, lane);
            }

            // ------------------------------ epilogue ------------------------------
            // Phase 1 (all warps): park the accumulators in the whole-tile staging buffer with the tile's own
            // row/column numbering (row = g*nb + i, col = (plane*wT + wl)*n + j).  Rows are stored in pairs:
            //     element (row, col)  ->  (row >> 1) * LD2 + (row & 1) * H + col,     H = 8 mod 16,  LD2 = 1 mod 16,
            // which makes the fragment-order stores here, the row loads and the column loads of phase 2 all
            // bank-conflict free (column loads 2-way when g*n is odd).
#if AFQMC_K2_ABLATE < 2
            mbar_wait(stg_free, tpar ^ 1u);                                    // previous tile has been read out
            if constexpr (MM > 0) {
#pragma unroll
                for (int m = 0; m < MM; ++m) {
                    const int row = (warp + m * WM) * 8 + (lane >> 2);
                    double *dst = staging + (row >> 1) * LD2 + (row & 1) * H + 2 * (lane & 3);
#pragma unroll
                    for (int q = 0; q < NT; ++q) { dst[q * 8] = acc[m][q][0]; dst[q * 8 + 1] = acc[m][q][1]; }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(stg_full);
            {
                // Phase 2 (all warps, once the whole tile is parked; the FP64 pipe is shared with the DMMAs, so these
                // DFMAs are only cheap while no warp is feeding it DMMAs): one (gamma g, walker wl) block
                // T = R + iI (n x n) per pass, lanes over j, loop over i:
                //     Re x += R_ij R_ji - I_ij I_ji,    Im x += 2 R_ij I_ji   (sum_ij I_ij R_ji = sum_ij R_ij I_ji by relabelling),
                //     t = sum_j T_jj.
                // When the tile has fewer blocks than warps, each block's i range is split into `rs` parts.
                const int g0 = rt * P.gT;
                const int gvalid = min(P.gT, P.n_gamma - g0);
                const int w0 = ct * P.wT;
                const int wvalid = min(P.wT, P.n_walkers - w0);
                const int planeoff = P.wT * n;
                const int nblk = gvalid * wvalid;
                const int rs = max(1, WM / nblk);
                double *redp = red + tpar * (K2_MAX_WT * K2_MAX_WM * 2);      // double-buffered by tile parity
                if (lane < K2_MAX_WT) { redp[(lane * K2_MAX_WM + warp) * 2] = 0.0; redp[(lane * K2_MAX_WM + warp) * 2 + 1] = 0.0; }
                mbar_wait(stg_full, tpar);
#if AFQMC_K2_ABLATE == 1
                for (int u = warp; u < 0; u += WM) {
#else
                for (int u = warp; u < nblk * rs; u += WM) {
#endif
                    const int blk = u / rs, part = u - blk * rs;
                    const int g = blk / wvalid, wl = blk - g * wvalid;
                    const int i_lo = (part * n) / rs, i_hi = ((part + 1) * n) / rs;
                    const int gn = g * P.nb, cb = wl * n;
                    const bool cplx = P.cplx != 0;
                    // element T_ij = R + iI of the block, from the parked products C = Ltilde theta^T:
                    //   real Ltilde:     R = C[i][re j],                   I = C[i][im j]
                    //   complex Ltilde:  R = C[re i][re j] - C[im i][im j], I = C[re i][im j] + C[im i][re j]   (rows im i = n + i)
                    auto elem = [&](const double *p, int row, int col, double &re, double &im) {
                        const double *q = p + (row >> 1) * LD2 + (row & 1) * H + col;
                        re = q[0]; im = q[planeoff];
                        if (cplx) {
                            const int r2 = row + n;
                            const double *q2 = p + (r2 >> 1) * LD2 + (r2 & 1) * H + col;
                            re -= q2[planeoff]; im += q2[0];
                        }
                    };
                    double xr = 0.0, xi = 0.0, yr = 0.0, yi = 0.0, tr = 0.0, ti = 0.0;
                    for (int j0 = 0; j0 < n; j0 += 32) {
                        const int j = j0 + lane;
                        if (j < n) {
                            const double *blkp = staging + cb;
                            if (part == 0) { double r, im; elem(blkp, gn + j, j, r, im); tr += r; ti += im; }
                            int i = i_lo;
                            for (; i + 1 < i_hi; i += 2) {                                          // two independent chains
                                double a_r, a_i, b_r, b_i, c_r, c_i, d_r, d_i;
                                elem(blkp, gn + i, j, a_r, a_i); elem(blkp, gn + j, i, b_r, b_i);            // T_ij, T_ji
                                elem(blkp, gn + i + 1, j, c_r, c_i); elem(blkp, gn + j, i + 1, d_r, d_i);
                                xr = fma(a_r, b_r, xr); yr = fma(c_r, d_r, yr);
                                xr = fma(-a_i, b_i, xr); yr = fma(-c_i, d_i, yr);
                                xi = fma(a_r, b_i, xi); yi = fma(c_r, d_i, yi);
                            }
                            if (i < i_hi) {
                                double a_r, a_i, b_r, b_i;
                                elem(blkp, gn + i, j, a_r, a_i); elem(blkp, gn + j, i, b_r, b_i);
                                xr = fma(a_r, b_r, xr);
                                xr = fma(-a_i, b_i, xr);
                                xi = fma(a_r, b_i, xi);
                            }
                        }
                    }
                    xr = warp_sum(xr + yr); xi = warp_sum(xi + yi);
                    if (part == 0) { tr = warp_sum(tr); ti = warp_sum(ti); }
                    if (lane == 0) {
                        if (part == 0) {
                            double *tp = P.tbuf + ((long long)(w0 + wl) * P.n_gamma + g0 + g) * 2;
                            tp[0] = tr; tp[1] = ti;
                        }
                        redp[(wl * K2_MAX_WM + warp) * 2] += xr;
                        redp[(wl * K2_MAX_WM + warp) * 2 + 1] += 2.0 * xi;
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(stg_free);
                if (warp == WM - 1) {                    // the lightest warp adds the per-warp shares in a fixed order
                    mbar_wait(stg_free, tpar);
                    if (lane < wvalid) {
                        double sr = 0.0, si = 0.0;
                        for (int q = 0; q < WM; ++q) { sr += redp[(lane * K2_MAX_WM + q) * 2]; si += redp[(lane * K2_MAX_WM + q) * 2 + 1]; }
                        double *xp = P.xpart + ((long long)rt * P.maxw + w0 + lane) * 2;
                        xp[0] = sr; xp[1] = si;
                    }
                }
            }
#else   // keep the products alive (ptxas would drop DMMAs whose results are never read)
            if constexpr (MM > 0) {
                double keep = 0.0;
#pragma unroll
                for (int m = 0; m < MM; ++m)
#pragma unroll
                    for (int q = 0; q < NT; ++q) keep += acc[m][q][0] + acc[m][q][1];
                if (keep == 1.2345678e300) P.tbuf[0] = keep;
            }
#endif  // AFQMC_K2_ABLATE < 2
            tpar ^= 1u;
            rt += step_rt; ct += step_ct;
            if (ct >= P.n_ct) { ct -= P.n_ct; ++rt; }
        }
    };
    if (my_mt == MT) run_tiles(std::integral_constant<int, MT>{});
    else run_tiles(std::integral_constant<int, MT - 1>{});
}

// ------------------------------------------------------------------------------------------------------------------
// Force-bias GEMM (Eq. 24; Listing 3): xbar^gamma_w = sum_ip Ltilde^gamma_ip theta^w_ip.
// Same operand ring and K loop as the exchange kernel, with the operands packed for n = 1 and k = (i, p): rows are
// gamma (x Re/Im of Ltilde for a complex trial), columns are (plane, walker), every warp owns one 8-row strip and all NT
// column blocks.  The K range is cut into `ksplit` equal parts so that (row tile, K part, column tile) items fill whole
// rounds of the persistent grid; every accumulator element is stored raw and `k4_force_bias_combine` adds the parts in
// a fixed order.
struct K2FbParams {
    const double *A, *B;           // packed operands (common.cuh), k-steps per tile = ksplit * kps
    long long itemA_doubles;       // one (row tile, K part) of A: kps * strips * 32
    long long tileB_doubles;       // one column tile of B, all K parts
    long long partB_doubles;       // one K part of a B tile: kps * NT * 32
    int rows_per_tile, rows_total; // valid rows per row tile, n_gamma * nb
    int strips, WM;
    int kps, ksc, nchunks, nstages;
    int n_items_r;                 // row tiles * ksplit
    int ksplit, n_ct;
    double *craw;                  // [ksplit][rows_total][n_ct][8 * NT]
};

template <int NT>
__global__ void __launch_bounds__(32 * K2_MAX_WM) k2_force_bias(const K2FbParams P) {
    extern __shared__ __align__(128) unsigned char k2_smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int WM = P.WM;
    const uint32_t a_chunk_bytes = (uint32_t)P.ksc * P.strips * 256u;
    const uint32_t b_chunk_bytes = (uint32_t)P.ksc * NT * 256u;
    const uint32_t stage_bytes = a_chunk_bytes + b_chunk_bytes;
    unsigned char *stage_base = k2_smem;
    uint64_t *full_bar = reinterpret_cast<uint64_t *>(k2_smem + (size_t)P.nstages * stage_bytes);
    uint64_t *empty_bar = full_bar + P.nstages;
    const int mma_warps = min(WM, P.strips);
    if (tid == 0) {
        for (int s = 0; s < P.nstages; ++s) {
            mbar_init(&full_bar[s], 1);
            mbar_init(&empty_bar[s], mma_warps);
        }
        mbar_fence_init();
    }
    __syncthreads();
    if (warp >= mma_warps) return;                       // no strip, no barrier duty

    const int step_rt = (int)(gridDim.x / (unsigned)P.n_ct), step_ct = (int)(gridDim.x % (unsigned)P.n_ct);
    const int first_rt = (int)(blockIdx.x / (unsigned)P.n_ct), first_ct = (int)(blockIdx.x % (unsigned)P.n_ct);

    const bool producer_warp = (warp == mma_warps - 1);
    int p_rt = first_rt, p_ct = first_ct, p_chunk = 0, p_stage = 0;
    uint32_t p_phase = 0;
    const double *p_a = P.A + (long long)p_rt * P.itemA_doubles;
    const double *p_b = P.B + (long long)p_ct * P.tileB_doubles + (p_rt % P.ksplit) * P.partB_doubles;
    auto produce_poll = [&]() {
        if (p_rt >= P.n_items_r) return;
        if (!mbar_test_addr(smem_u32(&empty_bar[p_stage]), p_phase ^ 1u)) return;
        mbar_arrive_expect_tx(&full_bar[p_stage], a_chunk_bytes + b_chunk_bytes);
        unsigned char *dst = stage_base + (size_t)p_stage * stage_bytes;
        bulk_g2s(dst, p_a, a_chunk_bytes, &full_bar[p_stage]);
        bulk_g2s(dst + a_chunk_bytes, p_b, b_chunk_bytes, &full_bar[p_stage]);
        p_a += a_chunk_bytes / 8; p_b += b_chunk_bytes / 8;
        if (++p_stage == P.nstages) { p_stage = 0; p_phase ^= 1u; }
        if (++p_chunk == P.nchunks) {
            p_chunk = 0;
            p_rt += step_rt; p_ct += step_ct;
            if (p_ct >= P.n_ct) { p_ct -= P.n_ct; ++p_rt; }
            p_a = P.A + (long long)p_rt * P.itemA_doubles;
            p_b = P.B + (long long)p_ct * P.tileB_doubles + (p_rt % P.ksplit) * P.partB_doubles;
        }
    };
    if (producer_warp && lane == 0)
        for (int d = 0; d < P.nstages; ++d) produce_poll();

    K2Ring R;
    R.smem_base = smem_u32(stage_base); R.stage_bytes = stage_bytes; R.a_chunk_bytes = a_chunk_bytes;
    R.a_kstride = (uint32_t)P.strips * 256u;
    R.full_bar = smem_u32(full_bar); R.empty_bar = smem_u32(empty_bar);
    R.nstages = P.nstages; R.ksc = P.ksc; R.nchunks = P.nchunks; R.last_ks = P.ksc; R.ksteps = P.kps;   // whole chunks only
    R.stage = 0; R.phase = 0;
    const uint32_t frag_off = (uint32_t)warp * 256u + 8u * lane;

    for (int rt = first_rt, ct = first_ct; rt < P.n_items_r;) {
        double acc[1][NT][2];
#pragma unroll
        for (int q = 0; q < NT; ++q) { acc[0][q][0] = 0.0; acc[0][q][1] = 0.0; }
        k2_tile_mma<1, NT>(acc, R, frag_off, 0u, producer_warp, produce_poll, lane);
        const int rtile = rt / P.ksplit, part = rt - rtile * P.ksplit;
        const int lrow = warp * 8 + (lane >> 2);
        const int row = rtile * P.rows_per_tile + lrow;
        if (lrow < P.rows_per_tile && row < P.rows_total) {
            double *dst = P.craw + (((long long)part * P.rows_total + row) * P.n_ct + ct) * (NT * 8) + 2 * (lane & 3);
#pragma unroll
            for (int q = 0; q < NT; ++q) *reinterpret_cast<double2 *>(dst + q * 8) = make_double2(acc[0][q][0], acc[0][q][1]);
        }
        rt += step_rt; ct += step_ct;
        if (ct >= P.n_ct) { ct -= P.n_ct; ++rt; }
    }
}

}  // namespace afqmc
