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
// phi is staged 32 rows at a time in a two-stage shared-memory ring by 16-byte asynchronous copies (LDGSTS) issued by
// all threads (per-row bulk copies from one warp were measured: their issue latency, not the data, set the pace); rows
// are padded to a pitch of 32 (mod 64) bytes, which makes both fragment patterns bank-conflict free.  The inverse is
// formed in shared memory by n exchange steps on an n x n ping-pong pair with ONE CTA barrier per step (k1_gauss_jordan
// below).  The first chunk of the theta pass is in flight during that phase.
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
    int w0;                       // walker of blockIdx.x == 0 (launches on a range of walkers)
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
    L.total = L.off_misc + 64 * 4 * 2 + 64 * 16 + 128 * 8 + 16 * 8 + 16;   // rowof, kof, pivots, keys, reductions
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

// 1 / x for a positive normal x: MUFU.RCP64H (about 20 bits) and two Newton steps.
__device__ __forceinline__ double fast_rcp(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;\n" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    y = fma(y, e, y);
    e = fma(-x, y, 1.0);
    return fma(y, e, y);
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

__device__ __forceinline__ void cp_async16(uint32_t dst_smem, const void *src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(dst_smem), "l"(src) : "memory");
}
__device__ __forceinline__ double2 lds_c128(uint32_t addr) {
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];\n" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts_c128(uint32_t addr, double2 v) {
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};\n" ::"r"(addr), "d"(v.x), "d"(v.y) : "memory");
}

// Pivot of step k when |a|^2 is zero, NaN or out of range: the unused row of largest |a_ik| by hypot().  Returns the
// row, or -1 when the column is exactly zero (or all NaN) below the used rows.  Warp-uniform result.
struct K1SlowPivot { double inv_re, inv_im; int row; };
__device__ __noinline__ K1SlowPivot k1_slow_pivot(uint32_t cur, int n, int k, unsigned long long used, int lane) {
    double m = -1.0;
    int r = 0x7fffffff;
    for (int i = lane; i < n; i += 32) {
        if (!((used >> i) & 1ull)) {
            const double2 c = lds_c128(cur + (uint32_t)(i * n + k) * 16u);
            const double h = hypot(c.x, c.y);
            if (h > m) { m = h; r = i; }
        }
    }
    warp_argmax(m, r);
    if (!(m > 0.0)) return K1SlowPivot{0.0, 0.0, -1};
    const double2 inv = crecip(lds_c128(cur + (uint32_t)(r * n + k) * 16u));
    return K1SlowPivot{inv.x, inv.y, r};
}

// X = S^-1 by n exchange steps (Gauss-Jordan, partial pivoting without row swaps), all THREADS threads of the CTA, one
// CTA barrier per step.  Step k with pivot row r (the unused row of largest |a_rk|), p = a_rk, q_j = a_rj / p (j != k), q_k = -1/p:
//     a_rj <- -q_j,        a_ij <- a_ij - a_ik q_j   (i != r; with a_ik taken as 0 on the left for j = k)
// i.e. a_rk <- 1/p, a_rj <- -a_rj/p, a_ik <- a_ik/p, a_ij <- a_ij - a_ik a_rj/p.  Afterwards X_ij = W[rowof[i]][kof[j]]
// and det S = sgn(k -> rowof[k]) prod_k p_k.  The matrix ping-pongs between w_start and w_other (shared-window addresses,
// [n][n] complex; the result is in w_start for even n, w_other for odd n).  2^LG threads span a matrix row, thread
// (ty, tx) keeps elements (ty + u RY, tx), u < ROWS, in registers for the whole elimination and re-publishes them every
// step; per step it reads only column k of its rows, the pivot and its element of the pivot row.  This phase is bound
// by instruction issue (four CTAs share an SM), so addresses are 32-bit shared-window offsets formed with one add, and
// the pivot search runs on integers: the thread that writes column k + 1 leaves |a|^2 in keys[], the warps mask the used
// rows and take the maximum of the bit patterns with three warp-wide integer reductions.
// Returns false if S is singular (a column is exactly zero below the used rows).  Not inlined: the loop then has the
// kernel's whole register budget to itself (the caller's live values are parked on the stack once, outside the loop).
template <int ROWS, int LG, int THREADS>
__device__ __noinline__ bool k1_gauss_jordan(const int n, const uint32_t w_start, const uint32_t w_other, const uint32_t keys_u,
                                                int *rowof, double2 *pivs, const int tid) {
    constexpr int RY = THREADS >> LG;
    const int lane = tid & 31, tx = tid & ((1 << LG) - 1), ty = tid >> LG;
    const bool col_ok = tx < n;
    const uint32_t txo = (col_ok ? tx : 0) * 16u;
    const uint32_t rowbase = (uint32_t)(ty * n) * 16u, rstep = (uint32_t)(RY * n) * 16u;
    double2 a[ROWS];
#pragma unroll
    for (int u = 0; u < ROWS; ++u) a[u] = (ty + u * RY < n) ? lds_c128(w_start + rowbase + u * rstep + txo) : make_double2(0.0, 0.0);
    uint32_t cur = w_start, nxt = w_other;
    unsigned long long used = 0ull;
    for (int k = 0; k < n; ++k) {
        const uint32_t koff = (uint32_t)k * 16u;
        const uint32_t kcur = keys_u + (k & 1) * 512u, knxt = keys_u + ((k + 1) & 1) * 512u;
        unsigned long long kb = 0ull;
        int row = lane;
        if (lane < n && !((used >> lane) & 1ull)) kb = (unsigned long long)__double_as_longlong(lds_f64_dyn(kcur + lane * 8));
        if (LG == 6 && lane + 32 < n && !((used >> (lane + 32)) & 1ull)) {
            const unsigned long long k2 = (unsigned long long)__double_as_longlong(lds_f64_dyn(kcur + (lane + 32) * 8));
            if (k2 > kb) { kb = k2; row = lane + 32; }
        }
        const unsigned hi = (unsigned)(kb >> 32), lo = (unsigned)kb;
        const unsigned mh = __reduce_max_sync(0xffffffffu, hi);
        const unsigned ml = __reduce_max_sync(0xffffffffu, hi == mh ? lo : 0u);
        int r = (int)__reduce_min_sync(0xffffffffu, (hi == mh && lo == ml) ? (unsigned)row : 0x7fffffffu);
        const double key = __hiloint2double((int)mh, (int)ml);
        double2 q, p;                                               // q_j = a_rj / p, q_k = -1 / p
        if (key > 1e-280 && key < 1e280) {
            const uint32_t prow = cur + (uint32_t)(r * n) * 16u;
            p = lds_c128(prow + koff);
            const double2 arj = lds_c128(prow + txo);
            const double d = fast_rcp(key);                         // key = |p|^2
            double2 t = make_double2(fma(arj.x, p.x, arj.y * p.y), fma(arj.y, p.x, -arj.x * p.y));   // a_rj conj(p)
            if (tx == k) t = make_double2(-p.x, p.y);
            q = make_double2(t.x * d, t.y * d);
        } else {
            const K1SlowPivot sp = k1_slow_pivot(cur, n, k, used, lane);
            r = sp.row;
            if (r < 0) return false;                                // uniform: every warp reads the same column
            const double2 inv = make_double2(sp.inv_re, sp.inv_im);
            const uint32_t prow = cur + (uint32_t)(r * n) * 16u;
            p = lds_c128(prow + koff);
            q = cmul(lds_c128(prow + txo), inv);
            if (tx == k) q = make_double2(-inv.x, -inv.y);
        }
        if (tid == 0) { rowof[k] = r; pivs[k] = p; }
        used |= 1ull << r;
        const bool kcol = tx == k, knext = tx == k + 1;
#pragma unroll
        for (int u = 0; u < ROWS; ++u) {
            const int i = ty + u * RY;
            if (i < n) {                                            // uniform per warp
                const double2 f = lds_c128(cur + rowbase + u * rstep + koff);    // column k (issued under the reciprocal above)
                double2 o = kcol ? make_double2(0.0, 0.0) : a[u];
                o.x = fma(-f.x, q.x, o.x); o.x = fma(f.y, q.y, o.x);
                o.y = fma(-f.x, q.y, o.y); o.y = fma(-f.y, q.x, o.y);
                if (i == r) o = make_double2(-q.x, -q.y);
                a[u] = o;
                if (col_ok) sts_c128(nxt + rowbase + u * rstep + txo, o);
                if (knext) asm volatile("st.shared.f64 [%0], %1;\n" ::"r"(knxt + (uint32_t)i * 8u), "d"(fma(o.x, o.x, o.y * o.y)) : "memory");
            }
        }
        __syncthreads();
        const uint32_t t = cur; cur = nxt; nxt = t;
    }
    return true;
}

// ---- K loops of the two products --------------------------------------------------------------------------------------
// A predicated-off DMMA still occupies the tensor pipe for its 16 cycles (measured: a kernel whose complex-trial DMMAs
// were compiled as @!P DMMA ran its S pass at twice the pipe time), so nothing in these loops is predicated: the number
// of column blocks a warp owns (CNT) and the complex-trial second product (CPLX) are template parameters, dispatched
// once per chunk by a warp-uniform branch.

// S pass, one chunk: nks k-steps.  pa: psi fragment of this warp's strip (+ im_off: Im psi), pb: B fragment of its first
// column block in the staged rows of phi, a_step / b_step: bytes per k-step.
template <int MAXT, int CNT, bool CPLX>
__device__ __forceinline__ void k1_s_kloop(double (&acc)[MAXT][2], uint32_t pa, uint32_t pb, const int nks, const uint32_t a_step,
                                           const uint32_t b_step, const uint32_t im_off, const bool odd_col) {
    for (int ks = 0; ks < nks; ++ks) {
        const double a = lds_f64_dyn(pa);
        double a2 = 0.0;
        if constexpr (CPLX) a2 = lds_f64_dyn(pa + im_off);
#pragma unroll
        for (int q = 0; q < CNT; ++q) {
            const double b = lds_f64_dyn(pb + q * 64);
            dmma_m8n8k4(acc[q][0], acc[q][1], a, b);
            if constexpr (CPLX) {     // + Im psi^T (phi_im, -phi_re): (a - ib)(x + iy) = (ax + by) + i(ay - bx)
                const double sw = lds_f64_dyn((pb + q * 64) ^ 8u);       // the other component of the same element
                dmma_m8n8k4(acc[q][0], acc[q][1], a2, odd_col ? -sw : sw);
            }
        }
        pa += a_step;
        pb += b_step;
    }
}
template <int MAXT, int CNT, bool CPLX>
__device__ __forceinline__ void k1_s_dispatch(const int cnt, double (&acc)[MAXT][2], uint32_t pa, uint32_t pb, const int nks,
                                              const uint32_t a_step, const uint32_t b_step, const uint32_t im_off, const bool odd_col) {
    if constexpr (CNT > 0) {
        if (cnt == CNT) k1_s_kloop<MAXT, CNT, CPLX>(acc, pa, pb, nks, a_step, b_step, im_off, odd_col);
        else k1_s_dispatch<MAXT, CNT - 1, CPLX>(cnt, acc, pa, pb, nks, a_step, b_step, im_off, odd_col);
    }
}

// theta pass, one chunk of one strip: kth k-steps.  pa: A fragment in the staged rows of phi, pb: this lane's component
// of the first column block's XF entry, b_step: bytes of XF per k-step, flip: sign-bit mask of the (re column, im row) lanes.
template <int MAXT, int CNT>
__device__ __forceinline__ void k1_t_kloop(double (&acc)[MAXT][2], uint32_t pa, uint32_t pb, const int kth, const uint32_t b_step,
                                           const int flip) {
    for (int ks = 0; ks < kth; ++ks) {
        const double a = lds_f64_dyn(pa);
#pragma unroll
        for (int q = 0; q < CNT; ++q) {
            double b = lds_f64_dyn(pb + q * 128);
            b = __hiloint2double(__double2hiint(b) ^ flip, __double2loint(b));
            dmma_m8n8k4(acc[q][0], acc[q][1], a, b);
        }
        pa += 32;
        pb += b_step;
    }
}
template <int MAXT, int CNT>
__device__ __forceinline__ void k1_t_dispatch(const int cnt, double (&acc)[MAXT][2], uint32_t pa, uint32_t pb, const int kth,
                                              const uint32_t b_step, const int flip) {
    if constexpr (CNT > 0) {
        if (cnt == CNT) k1_t_kloop<MAXT, CNT>(acc, pa, pb, kth, b_step, flip);
        else k1_t_dispatch<MAXT, CNT - 1>(cnt, acc, pa, pb, kth, b_step, flip);
    }
}

// Build with -DAFQMC_K1_PHASE_CLOCKS to accumulate, over all CTAs of all launches, the clock64() time from CTA start to
// each phase boundary (read back and reset with afqmc_k1_phase_clocks, which exists in such builds only): 1 ring
// cleared, 2 S pass done, 3 S stored, 4 inverse done, 5 XF done, 6 theta pass done, 7 end; entry 0 counts the CTAs.
#ifdef AFQMC_K1_PHASE_CLOCKS
__device__ unsigned long long g_k1_clocks[8];
#define K1_MARK(i)                                                                              \
    do {                                                                                        \
        if (threadIdx.x == 0) {                                                                 \
            if ((i) == 0) { k1_t0 = clock64(); atomicAdd(&g_k1_clocks[0], 1ull); }             \
            else atomicAdd(&g_k1_clocks[i], (unsigned long long)(clock64() - k1_t0));           \
        }                                                                                       \
    } while (0)
#else
#define K1_MARK(i) do { } while (0)
#endif

// SIZE 0: n <= 32 (<= 4 output tiles per warp and pass, 64 registers, four CTAs per SM); SIZE 1: n <= 64 with a shared-
// memory footprint that lets two CTAs share an SM (128 registers); SIZE 2: n <= 64, one CTA per SM (all registers).
template <int SIZE, bool WITH_FB>
__global__ void __launch_bounds__(K1_THREADS, SIZE == 0 ? 4 : SIZE == 1 ? 2 : 1) k1_overlap_inverse_theta(K1Params P) {
    constexpr bool BIG = SIZE > 0;
    constexpr int MAXT_S = BIG ? 16 : 4;     // S pass: tiles per warp
    constexpr int MAXT_T = BIG ? 8 : 4;      // theta pass: column blocks per warp
    const int w = blockIdx.x + P.w0, sp = blockIdx.y + P.spin0;
    const int n = P.n[sp], N = P.N;
    if (n == 0) return;
#ifdef AFQMC_K1_PHASE_CLOCKS
    long long k1_t0 = 0;
#endif
    K1_MARK(0);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const bool cplx = P.psiA_im[sp] != nullptr;
    const K1Layout L = k1_layout(n, cplx);
    extern __shared__ __align__(128) unsigned char k1_smem[];
    unsigned char *ring = k1_smem + L.off_ring;
    unsigned char *regA = k1_smem + L.off_a;
    int *rowof = reinterpret_cast<int *>(k1_smem + L.off_misc);        // [64] pivot row of step k
    int *kof = rowof + 64;                                               // [64] step at which row r was the pivot row
    double2 *pivs = reinterpret_cast<double2 *>(kof + 64);              // [64] pivots
    double *keys = reinterpret_cast<double *>(pivs + 64);               // [2][64] |a_ik|^2 of the unused rows: this step's column, next step's
    double *s_red = keys + 128;                                          // [16]

    const int nc = (N + K1_ROWS - 1) / K1_ROWS;                         // chunks per pass
    // Chunk c of either pass lives in ring stage c & 1; W0 shares stage 1, which the first chunk of the theta pass (in
    // flight during the inversion) does not use.
    double2 *W0 = reinterpret_cast<double2 *>(L.w0_in_ring ? ring + L.stage_bytes : k1_smem + L.off_w0);
    double2 *W1 = reinterpret_cast<double2 *>(regA);

    const double2 *phi = P.walkers + P.spin_off[sp] + (long long)w * N * n;   // [N][n]

    // The row pads of the ring must read as finite numbers (they meet zero operand entries): clear the ring once.
    for (int t = tid; t < 2 * L.stage_bytes / 16; t += K1_THREADS) reinterpret_cast<int4 *>(ring)[t] = make_int4(0, 0, 0, 0);
    __syncthreads();
    K1_MARK(1);

    // Staging: 16-byte asynchronous copies (LDGSTS) by all threads, thread (ty, tx) moves element tx of rows ty, ty + RY, ...
    // of the chunk into the padded rows of the stage; the psi fragments of an S chunk are contiguous.  One commit group
    // per chunk; the consumer waits for its own copies and then meets the others at the chunk's CTA barrier.
    const int c_lg = BIG ? 6 : 5, c_tx = tid & ((1 << c_lg) - 1), c_ty = tid >> c_lg, c_ry = K1_THREADS >> c_lg;
    const uint32_t ring_u = smem_u32(ring), a_u = smem_u32(regA);
    auto issue = [&](int c, bool with_psi) {
        const int r0 = c * K1_ROWS, rows = min(K1_ROWS, N - r0);
        if (c_tx < n) {
            const double2 *src = phi + (long long)r0 * n + c_tx;
            const uint32_t dst = ring_u + (c & 1) * L.stage_bytes + c_tx * 16;
            for (int r = c_ty; r < rows; r += c_ry) cp_async16(dst + r * L.pitch, src + (long long)r * n);
        }
        if (with_psi) {
            const int half16 = 8 * L.ns * 16;                  // 16-byte pieces of one plane of psi fragments per chunk
            const uint32_t dst = a_u + (c & 1) * L.psi_stage_bytes;
            const double2 *src = reinterpret_cast<const double2 *>(P.psiA[sp]) + (long long)c * half16;
            for (int t = tid; t < half16; t += K1_THREADS) cp_async16(dst + t * 16, src + t);
            if (cplx) {
                const double2 *src2 = reinterpret_cast<const double2 *>(P.psiA_im[sp]) + (long long)c * half16;
                for (int t = tid; t < half16; t += K1_THREADS) cp_async16(dst + (half16 + t) * 16, src2 + t);
            }
        }
        asm volatile("cp.async.commit_group;\n" ::: "memory");
    };
    issue(0, true);

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
        for (int g = 0; g < nc; ++g) {
            asm volatile("cp.async.wait_group 0;\n" ::: "memory");
            __syncthreads();                                    // chunk g has landed; stage (g + 1) & 1 has been read by every warp
            if (g + 1 < nc) issue(g + 1, true);
            if (s_cnt > 0) {
                const int rows = min(K1_ROWS, N - g * K1_ROWS), nks = (rows + 3) >> 2;
                uint32_t pa = a_u + (g & 1) * L.psi_stage_bytes + s_st * 256 + lane * 8;
                uint32_t pb = ring_u + (g & 1) * L.stage_bytes + fk * L.pitch + (8 * s_cb0 + fr) * 8;
                const uint32_t im_off = 8u * L.ns * 256u;
                if (cplx) k1_s_dispatch<MAXT_S, MAXT_S, true>(s_cnt, acc, pa, pb, nks, L.ns * 256, 4 * L.pitch, im_off, fr & 1);
                else k1_s_dispatch<MAXT_S, MAXT_S, false>(s_cnt, acc, pa, pb, nks, L.ns * 256, 4 * L.pitch, im_off, fr & 1);
            }
        }
        __syncthreads();                                        // the ring and the psi fragments are free
        K1_MARK(2);
        // C fragment: row lane / 4, columns 2 (lane % 4) + {0, 1} = (re, im) of j = 4 cb + lane % 4.  n odd: the result of
        // the n exchange steps must land in W0, so an odd n starts in W1.
        double2 *Ws = (n & 1) ? W1 : W0;
#pragma unroll
        for (int q = 0; q < MAXT_S; ++q) {
            if (q < s_cnt) {
                const int i = 8 * s_st + fr, j = 4 * (s_cb0 + q) + fk;
                if (i < n && j < n) Ws[i * n + j] = make_double2(acc[q][0], acc[q][1]);
                if (i < n && j == 0) keys[i] = fma(acc[q][0], acc[q][0], acc[q][1] * acc[q][1]);     // pivot search of step 0
            }
        }
    }
    issue(0, false);                                            // first chunk of the theta pass, lands during the inversion
    __syncthreads();
    K1_MARK(3);

    // ---- X = S^-1, result in W0 ------------------------------------------------------------------------------------------
    const bool singular = !k1_gauss_jordan<BIG ? 16 : 4, BIG ? 6 : 5, K1_THREADS>(n, smem_u32((n & 1) ? W1 : W0), smem_u32((n & 1) ? W0 : W1),
                                                                      smem_u32(keys), rowof, pivs, tid);
    K1_MARK(4);
    // ---- the fragment-ordered inverse XF -------------------------------------------------------
    // XF[(ks * ncb + cb) * 8 + (i & 1) * 4 + (j & 3)] = X_ij with ks = i >> 1, cb = j >> 2: the 8 complex numbers one B
    // fragment (k-step ks, column block cb) of the real image of X draws on, 128 contiguous bytes.
    if (!singular && tid < n) kof[rowof[tid]] = tid;
    __syncthreads();
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
    K1_MARK(5);

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
        const uint32_t xf_u = a_u;
        // B fragment lane (column c = lane / 4 -> (j, plane), k = lane % 4 -> (i, comp)): component comp ^ plane of
        // X_ij, negated where plane = re and comp = im   (theta_re = phi_re X_re - phi_im X_im, theta_im = phi_re X_im + phi_im X_re)
        const uint32_t b_lane = (uint32_t)(((fk >> 1) * 4 + (fr >> 1)) * 16 + (((fk & 1) ^ (fr & 1)) ? 8 : 0));
        const int flip = ((fr & 1) == 0 && (fk & 1) == 1) ? (int)0x80000000 : 0;
        for (int c = 0; c < nc; ++c) {
            asm volatile("cp.async.wait_group 0;\n" ::: "memory");
            __syncthreads();            // chunk c has landed; stage (c + 1) & 1 is free (c = 0: XF is complete and W0 is dead)
            if (c + 1 < nc) issue(c + 1, false);
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
                uint32_t pa = ring_u + (c & 1) * L.stage_bytes + (8 * t_s + fr) * L.pitch + fk * 8;
                uint32_t pb = xf_u + cb0 * 128 + b_lane;
                k1_t_dispatch<MAXT_T, MAXT_T>(cnt, acc, pa, pb, L.kth, L.ncb * 128, flip);
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
        }
    }

    K1_MARK(6);
    // ---- log det S = log(sgn prod_k p_k) and the block reduction of E1 (fixed order); outputs -----------------------------
    e1r = warp_sum(e1r);
    e1i = warp_sum(e1i);
    if (lane == 0) { s_red[2 * warp] = e1r; s_red[2 * warp + 1] = e1i; }
    double logabs = 0.0, argdet = 0.0;
    if (!singular && warp == 0) {
        // lane k: log|p_k|, arg p_k and whether k -> rowof[k] has an odd number of inversions behind k
        double la = 0.0, ang = 0.0;
        int inv = 0;
        for (int k = lane; k < n; k += 32) {
            const double2 p = pivs[k];
            const double m2 = fma(p.x, p.x, p.y * p.y);
            la += (m2 > 1e-280 && m2 < 1e280) ? 0.5 * log(m2) : log(hypot(p.x, p.y));
            ang += atan2(p.y, p.x);
            const int rk = rowof[k];
            for (int k2 = k + 1; k2 < n; ++k2) inv += rowof[k2] < rk;
        }
        la = warp_sum(la);
        ang = warp_sum(ang);
        if (__popc(__ballot_sync(0xffffffffu, inv & 1)) & 1) ang += CUDART_PI;     // sgn = (-1)^(number of inversions)
        ang -= 2.0 * CUDART_PI * rint(ang / (2.0 * CUDART_PI));                     // into [-pi, pi]
        if (ang <= -CUDART_PI) ang += 2.0 * CUDART_PI;
        logabs = la; argdet = ang;
    }
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
    K1_MARK(7);
}

}  // namespace afqmc
