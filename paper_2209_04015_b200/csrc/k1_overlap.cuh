// K1 -- per (walker, spin): overlap matrix, its inverse and determinant, theta, E1.
//   S      = psi^dagger phi                 (n x n)                          PAPER.md:143 (Eq. 16), Listing 2 line 1
//   log det S, X = S^-1   by Gauss-Jordan exchange steps with partial pivoting   PAPER.md:146-150 ("linalg.det"), Listing 2 line 2
//   theta  = (phi X)^T  (n x N), written as separate re / im planes           PAPER.md:191 (Eq. 23), Listing 2 line 3;
//            in K2's packed B-operand layout (common.cuh)                     re/im split: PAPER.md:260-262, 280
//   E1     = sum_jp htilde_jp theta_jp                                        PAPER.md:282 with Eq. 2, 22
// One CTA (8 warps) per (walker, spin).  Both products run on the FP64 tensor cores (DMMA.8x8x4):
//   S      real TN product  [n x N].[N x 2n]  : A = psi^T in fragment order (packed once by afqmc_create), B = the
//          interleaved (re, im) rows of phi exactly as they lie in memory;
//   theta  real product     [N x 2n].[2n x 2n]: A = the same rows of phi (k = (i, re/im)), B = the real image of X,
//          columns (j, re/im), read from a fragment-ordered copy of X with a sign flip on the (re column, im row) lanes.
// phi is staged 32 rows at a time in a two-stage shared-memory ring by per-row 1-D bulk async copies (TMA engine) that
// complete on an mbarrier; rows are padded to a pitch of 32 (mod 64) bytes, which makes both fragment patterns
// bank-conflict free.  The inverse is formed in shared memory by n exchange steps on an n x n ping-pong pair with ONE
// CTA barrier per step: every warp finds the pivot row itself (rows are never swapped: "implicit" pivoting), then all
// threads rewrite the matrix into the other buffer.  The first chunk of the theta pass is in flight during that phase.
#pragma once
#include <math_constants.h>
#include "common.cuh"

namespace afqmc {

constexpr int K1_THREADS = 256;
constexpr int K1_ROWS = 32;     // rows of phi per ring stage = 8 DMMA k-steps of S = 4 row strips of theta

struct K1Params {
    const double2 *walkers;       // alpha block [Nw][N][na], then beta block [Nw][N][nb]
    int n_walkers, N, maxw;
    int spin0;                    // spin of blockIdx.y == 0 (per-spin launches of the host-buffer entry point)
    int n[2];
    long long spin_off[2];        // offset of each spin block in `walkers`, in complex elements
    const double *psiA[2];        // Re psi^T as DMMA A fragments: [8 * chunks][strips][32], zero-padded
    const double *psiA_im[2];     // Im psi^T, same order, or nullptr for a real trial block
    const double *ht[2];          // [n][N] Re htilde
    const double *ht_im[2];       // Im htilde, or nullptr
    double *thetaB[2];            // packed B operand
    OperandLayout layB[2];
    double *thetaF[2];            // force-bias B operand (k = j * N + p, column = plane * wT + wl), or nullptr
    OperandLayout layF[2];
    double *logdet;               // [2][maxw][2]  (log|det|, arg)
    double *e1;                   // [2][maxw][2]
};

// Dynamic shared memory of one CTA (byte offsets).  Region A is, in turn, the psi fragment ring (S pass), the second
// Gauss-Jordan buffer W1, and the fragment-ordered inverse XF (theta pass).  W0 lies in the ring stage the first chunk
// of the theta pass does not use when it fits there (n <= 32 or so), which keeps four CTAs resident per SM.
struct K1Layout {
    int ns, ncb, kth;             // 8-row strips of S, 8-column blocks of (j, re/im), k-steps of the theta product
    int pitch, stage_bytes, psi_stage_bytes;
    int off_ring, off_w0, off_a, off_misc, total;
    bool w0_in_ring;
};
__host__ __device__ inline K1Layout k1_layout(int n, bool cplx) {
    K1Layout L;
    L.ns = (n + 7) / 8; L.ncb = (2 * n + 7) / 8; L.kth = (2 * n + 3) / 4;
    L.pitch = 32 * L.kth;                                   // >= 16 n, covers the zero-padded last k-step
    if (L.pitch % 64 == 0) L.pitch += 32;
    L.stage_bytes = K1_ROWS * L.pitch;
    L.psi_stage_bytes = 8 * L.ns * 256 * (cplx ? 2 : 1);
    const int w_bytes = 16 * n * n, xf_bytes = L.kth * L.ncb * 128;
    int a_bytes = 2 * L.psi_stage_bytes;
    if (w_bytes > a_bytes) a_bytes = w_bytes;
    if (xf_bytes > a_bytes) a_bytes = xf_bytes;
    L.w0_in_ring = w_bytes <= L.stage_bytes;
    L.off_ring = 0;
    L.off_w0 = 2 * L.stage_bytes;                           // only used when W0 does not fit a ring stage
    L.off_a = L.off_w0 + (L.w0_in_ring ? 0 : w_bytes);
    L.off_misc = L.off_a + a_bytes;
    L.total = L.off_misc + 64 * 4 * 2 + 64 * 16 + 16 * 8 + 2 * 8 + 16;   // rowof, kof, pivots, reductions, 2 mbarriers
    return L;
}

__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

// 1 / p for p != 0 without intermediate overflow or underflow.
__device__ __forceinline__ double2 crecip(double2 p) {
    const double s = fmax(fabs(p.x), fabs(p.y));
    double sc = 1.0;
    if (s < 1e-280) sc = 0x1p600; else if (s > 1e280) sc = 0x1p-600;
    const double x = p.x * sc, y = p.y * sc;
    const double d = 1.0 / (x * x + y * y);
    return make_double2(x * d * sc, -y * d * sc);
}

__device__ __forceinline__ double lds_f64_dyn(uint32_t addr) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];\n" : "=d"(v) : "r"(addr));
    return v;
}

// argmax over the warp of (key, row), ties to the lower row; keys are >= 0 or -1 (no candidate), never NaN.
__device__ __forceinline__ void warp_argmax(double &key, int &row) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double k2 = __shfl_xor_sync(0xffffffffu, key, o);
        const int r2 = __shfl_xor_sync(0xffffffffu, row, o);
        if (k2 > key || (k2 == key && r2 < row)) { key = k2; row = r2; }
    }
}

// BIG = false: n <= 32 (<= 4 output tiles per warp and pass, four CTAs per SM); BIG = true: n <= 64.
template <bool BIG, bool WITH_FB>
__global__ void __launch_bounds__(K1_THREADS, BIG ? 1 : 4) k1_overlap_inverse_theta(K1Params P) {
    constexpr int MAXT_S = BIG ? 16 : 4;     // S pass: tiles per warp
    constexpr int MAXT_T = BIG ? 8 : 4;      // theta pass: column blocks per warp
    const int w = blockIdx.x, sp = blockIdx.y + P.spin0;
    const int n = P.n[sp], N = P.N;
    if (n == 0) return;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const bool cplx = P.psiA_im[sp] != nullptr;
    const K1Layout L = k1_layout(n, cplx);
    extern __shared__ __align__(128) unsigned char k1_smem[];
    unsigned char *ring = k1_smem + L.off_ring;
    unsigned char *regA = k1_smem + L.off_a;
    int *rowof = reinterpret_cast<int *>(k1_smem + L.off_misc);        // [64] pivot row of step k
    int *kof = rowof + 64;                                               // [64] step at which row r was the pivot row
    double2 *pivs = reinterpret_cast<double2 *>(kof + 64);              // [64] pivots
    double *s_red = reinterpret_cast<double *>(pivs + 64);              // [16]
    uint64_t *full = reinterpret_cast<uint64_t *>(s_red + 16);          // [2]

    const int nc = (N + K1_ROWS - 1) / K1_ROWS;                         // chunks per pass
    const int st_w0 = (nc + 1) & 1;                                     // ring stage the first theta chunk does not use
    double2 *W0 = reinterpret_cast<double2 *>(L.w0_in_ring ? ring + st_w0 * L.stage_bytes : k1_smem + L.off_w0);
    double2 *W1 = reinterpret_cast<double2 *>(regA);

    const double2 *phi = P.walkers + P.spin_off[sp] + (long long)w * N * n;   // [N][n]
    const uint32_t row_bytes = 16u * n;

    // The row pads of the ring must read as finite numbers (they meet zero operand entries): clear the ring once.
    for (int t = tid; t < 2 * L.stage_bytes / 16; t += K1_THREADS) reinterpret_cast<int4 *>(ring)[t] = make_int4(0, 0, 0, 0);
    if (tid == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        mbar_fence_init();
    }
    asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
    __syncthreads();

    // Chunk g of the kernel (S pass: g = 0 .. nc-1, theta pass: g = nc .. 2 nc - 1) lives in stage g & 1; the stage's
    // barrier completes its (g >> 1)-th phase when the copies have landed.  Issued by warp 0, one row per lane.
    auto issue = [&](int g) {
        const int c = g < nc ? g : g - nc, stage = g & 1;
        const int r0 = c * K1_ROWS, rows = min(K1_ROWS, N - r0);
        const uint32_t psi_bytes = g < nc ? (uint32_t)L.psi_stage_bytes : 0u;
        if (lane == 0) mbar_arrive_expect_tx(&full[stage], rows * row_bytes + psi_bytes);
        __syncwarp();
        if (lane < rows) bulk_g2s(ring + stage * L.stage_bytes + lane * L.pitch, phi + (long long)(r0 + lane) * n, row_bytes, &full[stage]);
        if (g < nc && lane == 0) {
            const uint32_t half = 8u * L.ns * 256u;
            unsigned char *dst = regA + stage * L.psi_stage_bytes;
            bulk_g2s(dst, P.psiA[sp] + (long long)c * (half / 8), half, &full[stage]);
            if (cplx) bulk_g2s(dst + half, P.psiA_im[sp] + (long long)c * (half / 8), half, &full[stage]);
        }
    };
    if (warp == 0) {
        issue(0);
        if (nc > 1) issue(1);
    }

    // ---- S = psi^dagger phi = (Re psi - i Im psi)^T phi ---------------------------------------------------------------
    // Output tiles: 8-row strips st of i x 8-column blocks cb of (j, re/im).  n <= 32: warp -> (strip warp % ns, one of
    // 8 / ns groups of column blocks), so every SM sub-partition carries the same load; n > 32: warp = strip, all blocks.
    const int fr = lane >> 2, fk = lane & 3;
    {
        int s_st, s_cb0, s_cnt;
        if (BIG) {
            s_st = warp; s_cb0 = 0; s_cnt = warp < L.ns ? L.ncb : 0;
        } else {
            const int groups = 8 / L.ns, per = (L.ncb + groups - 1) / groups, grp = warp / L.ns;
            s_st = warp - grp * L.ns; s_cb0 = grp * per;
            s_cnt = grp < groups ? max(0, min(per, L.ncb - s_cb0)) : 0;
        }
        double acc[MAXT_S][2];
#pragma unroll
        for (int q = 0; q < MAXT_S; ++q) { acc[q][0] = 0.0; acc[q][1] = 0.0; }
        const uint32_t ring_u = smem_u32(ring), a_u = smem_u32(regA);
        for (int g = 0; g < nc; ++g) {
            mbar_wait(&full[g & 1], (g >> 1) & 1);
            if (s_cnt > 0) {
                const int rows = min(K1_ROWS, N - g * K1_ROWS), nks = (rows + 3) >> 2;
                uint32_t pa = a_u + (g & 1) * L.psi_stage_bytes + s_st * 256 + lane * 8;
                uint32_t pb = ring_u + (g & 1) * L.stage_bytes + fk * L.pitch + (8 * s_cb0 + fr) * 8;
                const uint32_t im_off = 8u * L.ns * 256u;
                for (int ks = 0; ks < nks; ++ks) {
                    const double a = lds_f64_dyn(pa);
                    const double a2 = cplx ? lds_f64_dyn(pa + im_off) : 0.0;
#pragma unroll
                    for (int q = 0; q < MAXT_S; ++q) {
                        if (q < s_cnt) {
                            const double b = lds_f64_dyn(pb + q * 64);
                            dmma_m8n8k4(acc[q][0], acc[q][1], a, b);
                            if (cplx) {    // + Im psi^T (phi_im, -phi_re): (a - ib)(x + iy) = (ax + by) + i(ay - bx)
                                const double sw = lds_f64_dyn((pb + q * 64) ^ 8u);     // the other component of the same element
                                dmma_m8n8k4(acc[q][0], acc[q][1], a2, (fr & 1) ? -sw : sw);
                            }
                        }
                    }
                    pa += L.ns * 256;
                    pb += 4 * L.pitch;
                }
            }
            __syncthreads();                                    // stage g & 1 has been read by every warp
            if (warp == 0 && g + 2 < nc) issue(g + 2);
        }
        // C fragment: row lane / 4, columns 2 (lane % 4) + {0, 1} = (re, im) of j = 4 cb + lane % 4.  n odd: the result of
        // the n exchange steps must land in W0, so an odd n starts in W1.
        double2 *Ws = (n & 1) ? W1 : W0;
#pragma unroll
        for (int q = 0; q < MAXT_S; ++q) {
            if (q < s_cnt) {
                const int i = 8 * s_st + fr, j = 4 * (s_cb0 + q) + fk;
                if (i < n && j < n) Ws[i * n + j] = make_double2(acc[q][0], acc[q][1]);
            }
        }
    }
    if (warp == 0) issue(nc);                                   // first chunk of the theta pass, lands during the inversion
    __syncthreads();

    // ---- X = S^-1 by n exchange steps (Gauss-Jordan, partial pivoting without row swaps) -----------------------------
    // Step k with pivot row r (the unused row of largest |a_rk|), p = a_rk:
    //     a_rk <- 1/p,   a_rj <- -a_rj / p,   a_ik <- a_ik / p,   a_ij <- a_ij - a_ik a_rj / p        (i != r, j != k)
    // Afterwards X_ij = W[rowof[i]][kof[j]] and det S = sgn(k -> rowof[k]) prod_k p_k.
    bool singular = false;
    {
        const int lg = BIG ? 6 : 5;
        const int tx = tid & ((1 << lg) - 1), ty = tid >> lg, RY = K1_THREADS >> lg;
        unsigned long long used = 0ull;
        double2 *cur = (n & 1) ? W1 : W0, *nxt = (n & 1) ? W0 : W1;
        for (int k = 0; k < n; ++k) {
            double key = -1.0;
            int row = 0x7fffffff;
            for (int i = lane; i < n; i += 32) {
                if (!((used >> i) & 1ull)) {
                    const double2 a = cur[i * n + k];
                    const double m = a.x * a.x + a.y * a.y;
                    if (m > key) { key = m; row = i; }
                }
            }
            warp_argmax(key, row);
            if (!(key > 1e-280 && key < 1e280)) {               // |a|^2 may have under- or overflowed: decide on |a| itself
                key = -1.0; row = 0x7fffffff;
                for (int i = lane; i < n; i += 32) {
                    if (!((used >> i) & 1ull)) {
                        const double2 a = cur[i * n + k];
                        const double m = hypot(a.x, a.y);
                        if (m > key) { key = m; row = i; }
                    }
                }
                warp_argmax(key, row);
            }
            if (!(key > 0.0)) { singular = true; break; }       // uniform: every warp reads the same column
            const int r = row;
            const double2 p = cur[r * n + k];
            const double2 inv = crecip(p);
            if (tid == 0) { rowof[k] = r; pivs[k] = p; }
            used |= 1ull << r;
            if (tx < n) {
                const double2 q = cmul(cur[r * n + tx], inv);
                for (int i = ty; i < n; i += RY) {
                    double2 o;
                    if (i == r) {
                        o = (tx == k) ? inv : make_double2(-q.x, -q.y);
                    } else {
                        const double2 f = cur[i * n + k];
                        if (tx == k) {
                            o = cmul(f, inv);
                        } else {
                            o = cur[i * n + tx];
                            o.x = fma(-f.x, q.x, o.x); o.x = fma(f.y, q.y, o.x);
                            o.y = fma(-f.x, q.y, o.y); o.y = fma(-f.y, q.x, o.y);
                        }
                    }
                    nxt[i * n + tx] = o;
                }
            }
            __syncthreads();
            double2 *t = cur; cur = nxt; nxt = t;
        }
    }

    // ---- log det S (warp 0) and the fragment-ordered inverse XF -------------------------------------------------------
    // XF[(ks * ncb + cb) * 8 + (i & 1) * 4 + (j & 3)] = X_ij with ks = i >> 1, cb = j >> 2: the 8 complex numbers one B
    // fragment (k-step ks, column block cb) of the real image of X draws on, 128 contiguous bytes.
    double logabs = 0.0, argdet = 0.0;
    if (!singular) {
        if (tid < n) kof[rowof[tid]] = tid;
        if (warp == 0) {
            double la = 0.0, pr = 1.0, pi = 0.0;
            for (int k = lane; k < n; k += 32) {
                const double2 p = pivs[k];
                const double m = hypot(p.x, p.y);
                la += log(m);
                const double2 u = cmul(make_double2(pr, pi), make_double2(p.x / m, p.y / m));
                pr = u.x; pi = u.y;
            }
            la = warp_sum(la);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const double r2 = __shfl_xor_sync(0xffffffffu, pr, o), i2 = __shfl_xor_sync(0xffffffffu, pi, o);
                const double2 u = cmul(make_double2(pr, pi), make_double2(r2, i2));
                pr = u.x; pi = u.y;
            }
            if (lane == 0) {                                    // parity of the permutation k -> rowof[k] by its cycles
                unsigned long long seen = 0ull;
                bool odd = false;
                for (int s = 0; s < n; ++s) {
                    if ((seen >> s) & 1ull) continue;
                    int len = 0;
                    for (int t = s; !((seen >> t) & 1ull); t = rowof[t]) { seen |= 1ull << t; ++len; }
                    odd ^= ((len & 1) == 0);
                }
                if (odd) { pr = -pr; pi = -pi; }
                logabs = la; argdet = atan2(pi, pr);
            }
        }
        __syncthreads();
    }
    {
        double2 *XF = reinterpret_cast<double2 *>(regA);
        const int slots = L.kth * L.ncb * 8;
        for (int e = tid; e < slots; e += K1_THREADS) {
            const int blk = e >> 3, ks = blk / L.ncb, cb = blk - ks * L.ncb;
            const int i = 2 * ks + ((e >> 2) & 1), j = 4 * cb + (e & 3);
            double2 v = make_double2(0.0, 0.0);
            if (i < n && j < n) v = singular ? make_double2(CUDART_NAN, CUDART_NAN) : W0[rowof[i] * n + kof[j]];
            XF[e] = v;
        }
    }
    asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");     // W0's ring stage is about to be refilled by bulk copies
    __syncthreads();
    if (warp == 0 && nc > 1) issue(nc + 1);

    // ---- theta_jp = sum_i phi_pi X_ij ; packed write; E1 partial ----------------------------------------------------------
    // Per chunk: warp -> (row strip warp & 3 of the chunk, half warp >> 2 of the column blocks).  C fragment: row p,
    // columns (re, im) of j = 4 cb + lane % 4.
    const OperandLayout lay = P.layB[sp];
    const int wT = lay.per_tile;
    const int tile = w / wT, wl = w - tile * wT;
    const int col_re = wl * n, col_im = (wT + wl) * n;
    double *out = P.thetaB[sp] + (long long)tile * lay.tile_doubles;
    const OperandLayout layF = P.layF[sp];
    double *outF = nullptr;
    int colF_re = 0, colF_im = 0;
    if (WITH_FB) {
        const int tileF = w / layF.per_tile, wlF = w - tileF * layF.per_tile;
        outF = P.thetaF[sp] + (long long)tileF * layF.tile_doubles;
        colF_re = wlF; colF_im = layF.per_tile + wlF;
    }
    const double *ht = P.ht[sp];
    const double *ht_im = P.ht_im[sp];
    double e1r = 0.0, e1i = 0.0;
    {
        const int t_s = warp & 3, half = warp >> 2;
        const int per = (L.ncb + 1) >> 1, cb0 = half * per, cnt = max(0, min(per, L.ncb - cb0));
        const uint32_t ring_u = smem_u32(ring), xf_u = smem_u32(regA);
        // B fragment lane (column c = lane / 4 -> (j, plane), k = lane % 4 -> (i, comp)): component comp ^ plane of
        // X_ij, negated where plane = re and comp = im   (theta_re = phi_re X_re - phi_im X_im, theta_im = phi_re X_im + phi_im X_re)
        const uint32_t b_lane = (uint32_t)(((fk >> 1) * 4 + (fr >> 1)) * 16 + (((fk & 1) ^ (fr & 1)) ? 8 : 0));
        const int flip = ((fr & 1) == 0 && (fk & 1) == 1) ? (int)0x80000000 : 0;
        for (int c = 0; c < nc; ++c) {
            const int g = nc + c;
            mbar_wait(&full[g & 1], (g >> 1) & 1);
            const int p = c * K1_ROWS + 8 * t_s + fr;
            if (c * K1_ROWS + 8 * t_s < N && cnt > 0) {
                double hv[MAXT_T], hi[MAXT_T];
#pragma unroll
                for (int q = 0; q < MAXT_T; ++q) {
                    const int j = 4 * (cb0 + q) + fk;
                    const bool ok = q < cnt && p < N && j < n;
                    hv[q] = ok ? ht[(long long)j * N + p] : 0.0;
                    hi[q] = (ok && cplx) ? ht_im[(long long)j * N + p] : 0.0;
                }
                double acc[MAXT_T][2];
#pragma unroll
                for (int q = 0; q < MAXT_T; ++q) { acc[q][0] = 0.0; acc[q][1] = 0.0; }
                uint32_t pa = ring_u + (g & 1) * L.stage_bytes + (8 * t_s + fr) * L.pitch + fk * 8;
                uint32_t pb = xf_u + cb0 * 128 + b_lane;
                for (int ks = 0; ks < L.kth; ++ks) {
                    const double a = lds_f64_dyn(pa);
#pragma unroll
                    for (int q = 0; q < MAXT_T; ++q) {
                        if (q < cnt) {
                            double b = lds_f64_dyn(pb + q * 128);
                            b = __hiloint2double(__double2hiint(b) ^ flip, __double2loint(b));
                            dmma_m8n8k4(acc[q][0], acc[q][1], a, b);
                        }
                    }
                    pa += 32;
                    pb += L.ncb * 128;
                }
                if (p < N) {
                    const long long prow = (long long)(p >> 2) * lay.strips * 32 + (p & 3);
#pragma unroll
                    for (int q = 0; q < MAXT_T; ++q) {
                        const int j = 4 * (cb0 + q) + fk;
                        if (q < cnt && j < n) {
                            const double tr = acc[q][0], ti = acc[q][1];
                            e1r = fma(hv[q], tr, e1r);
                            e1i = fma(hv[q], ti, e1i);
                            if (cplx) { e1r = fma(-hi[q], ti, e1r); e1i = fma(hi[q], tr, e1i); }
                            const int cr = col_re + j, ci = col_im + j;
                            out[prow + (cr >> 3) * 32 + (cr & 7) * 4] = tr;
                            out[prow + (ci >> 3) * 32 + (ci & 7) * 4] = ti;
                            if (WITH_FB) {
                                const long long kk = (long long)j * N + p;
                                const long long krow = (kk >> 2) * layF.strips * 32 + (kk & 3);
                                outF[krow + (colF_re >> 3) * 32 + (colF_re & 7) * 4] = tr;
                                outF[krow + (colF_im >> 3) * 32 + (colF_im & 7) * 4] = ti;
                            }
                        }
                    }
                }
            }
            __syncthreads();
            if (warp == 0 && c + 2 < nc) issue(g + 2);
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
            ld[0] = logabs; ld[1] = argdet;
        }
    }
}

}  // namespace afqmc
