// EXPERIMENT -- Ozaki-scheme FP64 emulation of the contraction of PAPER.md:237-242 (Eq. 29),
//     T = Ltilde theta^T ,   i.e. a real GEMM  C[M x Ncol] = A[M x K] B[Ncol x K]^T  with K = N orbitals,
// on the 5th-generation tensor cores (tcgen05.mma kind::i8, accumulators in TMEM), stand-alone: its own shared library
// (libafqmc_ozaki.so, include/afqmc_ozaki.h), not on the product path.  FP64 has no tcgen05 kind, so this is the only
// route in this project past the 64 FMA/clk/SM FP64 issue limit that K2 (DMMA.8x8x4) sits at.
//
// Scheme.  Every row of A and of B is scaled by a power of two so that |x| < 1/2 and cut into `slices` signed 7-bit digits
//     x = 2^E sum_s a_s 2^(-7 (s + 1)) + tail ,   a_s = rint(r_s) in [-64, 64],  r_(s+1) = 128 (r_s - a_s)     (exact in FP64)
// so that  C_ij = 2^(EA_i + EB_j) sum_d 2^(-7 (d + 2)) S_d ,   S_d = sum_(s + t = d) A_s B_t^T  (exact INT32: K 64^2 (d+1) < 2^31).
// All slice products of one weight class d accumulate in the SAME TMEM accumulator, so the epilogue converts `slices`
// integers per output element instead of slices (slices + 1) / 2.  Keeping s + t < slices leaves a relative truncation
// of about K 2^(-7 slices) against max|a_i| max|b_j|.
//
// Kernel structure (B200): persistent CTAs, one per SM; warp 0 = TMA producer (1-D bulk copies of pre-packed core-matrix
// blocks into a 4-stage ring), warp 1 = MMA issuer (one elected lane, UTCIMMA 128 x 64 x 32), warps 2..5 = epilogue
// (tcgen05.ld, INT32 -> FP64, scaling, optional store, checksum).  Operands are library-owned, hence packed directly
// in the canonical K-major no-swizzle UMMA layout (8-row x 16-byte core matrices): no tensor maps needed.
// Every mbarrier wait is bounded: on a time-out the kernel sets an error flag and all roles leave.
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <string>

#include "../../include/afqmc_ozaki.h"

namespace {

constexpr int BM = 128, BN = 64, BK = 32;          // UTCIMMA shape: 128 x 64 x 32 int8
constexpr int MAX_SLICES = 8;                      // 8 weight classes x 64 columns = the 512 TMEM columns
constexpr int STAGES = 4;
constexpr int A_SLICE_BYTES = BM * BK, B_SLICE_BYTES = BN * BK;
constexpr int THREADS = 192;                       // producer warp, MMA warp, 4 epilogue warps
constexpr long long WAIT_CYCLES = 4000000000LL;    // ~2 s

thread_local std::string g_err;

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try(uint64_t *bar, uint32_t parity) {
    uint32_t ok;
    asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}\n"
                 : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0;
}
// Bounded wait: false (and *err = code) if the barrier does not complete within WAIT_CYCLES or another role has failed.
__device__ __forceinline__ bool mbar_wait_bounded(uint64_t *bar, uint32_t parity, volatile int *err, int code) {
    const long long t0 = clock64();
    while (!mbar_try(bar, parity)) {
        if (*err != 0) return false;
        if (clock64() - t0 > WAIT_CYCLES) { *err = code; return false; }
    }
    return true;
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// K-major, no swizzle: core matrix = 8 rows x 16 bytes (128 contiguous bytes); LBO = byte distance between the two
// 16-byte K halves of one MMA, SBO = byte distance between 8-row groups (both >> 4); descriptor version 1 (sm_100).
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo) {
    return (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)((lbo >> 4) & 0x3FFF) << 16) | ((uint64_t)((sbo >> 4) & 0x3FFF) << 32) |
           (1ULL << 46);
}
__device__ __forceinline__ void umma_i8(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
    asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n}\n" ::"r"(tmem_d),
                 "l"(da), "l"(db), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t *bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];\n"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
          "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]),
          "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]),
          "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory");
}

// ---- slicing: one warp per row of X [R][K] (row pitch ld) ---------------------------------------------------------------
// packed[tile][kstep][slice][k16][row group][8 rows][16 bytes], tile = `tile_rows` rows; scale[row] = 2^E.
__global__ void oz_slice(const double *__restrict__ X, long long ld, int R, int K, int nk, int slices, int tile_rows,
                         int8_t *__restrict__ packed, double *__restrict__ scale) {
    const int lane = threadIdx.x & 31, row = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (row >= R) return;
    const double *x = X + (long long)row * ld;
    double m = 0.0;
    for (int k = lane; k < K; k += 32) m = fmax(m, fabs(x[k]));
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    int e = 0;
    if (m > 0.0) frexp(m, &e);
    const int E = e + 1;                                  // |x| 2^-E < 1/2
    if (lane == 0) scale[row] = ldexp(1.0, E);
    const int tile = row / tile_rows, rin = row - tile * tile_rows, groups = tile_rows / 8;
    for (int k = lane; k < nk * 32; k += 32) {
        double r = k < K ? ldexp(x[k], -E) : 0.0;
        const int ks = k >> 5, k16 = (k >> 4) & 1, byte = k & 15;
        for (int s = 0; s < slices; ++s) {
            r *= 128.0;
            const double a = rint(r);
            r -= a;
            const long long off = (((((long long)tile * nk + ks) * slices + s) * 2 + k16) * groups + (rin >> 3)) * 128 + (rin & 7) * 16 + byte;
            packed[off] = (int8_t)(int)a;
        }
    }
}

struct OzParams {
    const int8_t *A, *B;              // packed slices
    const double *scaleA, *scaleB;    // 2^E per row / column
    int M, Ncol, nk, slices, n_rt, n_ct;
    double *C;                        // [M][ldc] or nullptr
    long long ldc;
    double *checksum;                 // sum of C^2 over everything (atomicAdd)
    int *err;
};

__global__ void __launch_bounds__(THREADS, 1) oz_gemm(const OzParams P) {
    extern __shared__ __align__(1024) unsigned char smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int a_bytes = P.slices * A_SLICE_BYTES, b_bytes = P.slices * B_SLICE_BYTES, stage_bytes = a_bytes + b_bytes;
    __shared__ uint64_t full_bar[STAGES], empty_bar[STAGES], acc_full, acc_empty;
    __shared__ uint32_t tmem_base_s;
    volatile int *err = P.err;
    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); }
        mbar_init(&acc_full, 1);
        mbar_init(&acc_empty, 4);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    if (warp == 1) {                                       // the MMA warp owns the TMEM allocation
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;\n" ::"r"(smem_u32(&tmem_base_s)));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n");
    }
    asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
    const uint32_t tmem_base = tmem_base_s;
    const long long n_tiles = (long long)P.n_rt * P.n_ct;

    if (warp == 0) {
        // ------------------------------- TMA producer -------------------------------
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            bool ok = true;
            for (long long t = blockIdx.x; t < n_tiles && ok; t += gridDim.x) {
                const int rt = (int)(t / P.n_ct), ct = (int)(t - (long long)rt * P.n_ct);
                for (int ks = 0; ks < P.nk; ++ks) {
                    if (!(ok = mbar_wait_bounded(&empty_bar[stage], phase ^ 1u, err, 1))) break;
                    unsigned char *dst = smem + (size_t)stage * stage_bytes;
                    mbar_expect_tx(&full_bar[stage], (uint32_t)stage_bytes);
                    bulk_g2s(dst, P.A + ((long long)rt * P.nk + ks) * a_bytes, (uint32_t)a_bytes, &full_bar[stage]);
                    bulk_g2s(dst + a_bytes, P.B + ((long long)ct * P.nk + ks) * b_bytes, (uint32_t)b_bytes, &full_bar[stage]);
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        // ------------------------------- MMA issuer -------------------------------
        if (lane == 0) {
            // instruction descriptor: D = S32 (2 << 4), A = B = signed 8 bit (1 << 7, 1 << 10), both K-major, N >> 3 at bit 17, M >> 4 at bit 24
            const uint32_t idesc = (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(BN >> 3) << 17) | ((uint32_t)(BM >> 4) << 24);
            int stage = 0;
            uint32_t phase = 0, tphase = 0;
            bool ok = true;
            for (long long t = blockIdx.x; t < n_tiles && ok; t += gridDim.x) {
                if (!(ok = mbar_wait_bounded(&acc_empty, tphase ^ 1u, err, 2))) break;      // epilogue has drained TMEM
                asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
                for (int ks = 0; ks < P.nk; ++ks) {
                    if (!(ok = mbar_wait_bounded(&full_bar[stage], phase, err, 3))) break;
                    asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
                    const uint32_t sa = smem_u32(smem + (size_t)stage * stage_bytes), sb = sa + a_bytes;
                    for (int d = 0; d < P.slices; ++d) {                                  // weight class d = s + t
                        for (int s = 0; s <= d; ++s) {
                            const uint64_t da = umma_desc(sa + s * A_SLICE_BYTES, (BM / 8) * 128, 128);
                            const uint64_t db = umma_desc(sb + (d - s) * B_SLICE_BYTES, (BN / 8) * 128, 128);
                            umma_i8(tmem_base + d * BN, da, db, idesc, (ks > 0 || s > 0) ? 1u : 0u);
                        }
                    }
                    umma_commit(&empty_bar[stage]);                                       // stage free once these MMAs have read it
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
                if (ok) umma_commit(&acc_full);                                           // accumulators complete
                tphase ^= 1u;
            }
        }
    } else {
        // ------------------------------- epilogue: warps 2..5, TMEM lane quarter = warp % 4 -------------------------------
        const int q = warp & 3;
        uint32_t tphase = 0;
        double csum = 0.0;
        bool ok = true;
        for (long long t = blockIdx.x; t < n_tiles && ok; t += gridDim.x) {
            const int rt = (int)(t / P.n_ct), ct = (int)(t - (long long)rt * P.n_ct);
            if (!(ok = mbar_wait_bounded(&acc_full, tphase, err, 4))) break;
            asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
            const int row = rt * BM + q * 32 + lane;
            const double sa = row < P.M ? P.scaleA[row] : 0.0;
#pragma unroll 1
            for (int h = 0; h < BN / 32; ++h) {
                double acc[32];
#pragma unroll
                for (int c = 0; c < 32; ++c) acc[c] = 0.0;
                double wd = 1.0 / 16384.0;                                                 // 2^(-7 (d + 2)), d = 0
                for (int d = 0; d < P.slices; ++d) {
                    uint32_t r[32];
                    tmem_ld32(tmem_base + ((uint32_t)(q * 32) << 16) + d * BN + h * 32, r);
#pragma unroll
                    for (int c = 0; c < 32; ++c) acc[c] = fma((double)(int)r[c], wd, acc[c]);
                    wd *= 1.0 / 128.0;
                }
                const int col0 = ct * BN + h * 32;
#pragma unroll
                for (int c = 0; c < 32; ++c) {
                    const int col = col0 + c;
                    const double v = (col < P.Ncol) ? acc[c] * sa * P.scaleB[col] : 0.0;
                    csum = fma(v, v, csum);
                    if (P.C && row < P.M && col < P.Ncol) P.C[(long long)row * P.ldc + col] = v;
                }
            }
            asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
            __syncwarp();
            if (lane == 0) mbar_arrive(&acc_empty);
            tphase ^= 1u;
        }
        for (int o = 16; o > 0; o >>= 1) csum += __shfl_xor_sync(0xffffffffu, csum, o);
        if (lane == 0 && P.checksum) atomicAdd(P.checksum, csum);
    }
    __syncthreads();
    if (warp == 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;\n" ::"r"(tmem_base));
}

int fail(int code, const char *msg) { g_err = msg; return code; }

}  // namespace

extern "C" {

const char *afqmc_ozaki_last_error(void) { return g_err.c_str(); }

int afqmc_ozaki_gemm(const double *A, const double *B, int M, int Ncol, int K, int slices, double *C, double *checksum,
                     float *ms_slice, float *ms_gemm, int repeats, void *stream_) {
    if (!A || !B || M < 1 || Ncol < 1 || K < 1 || slices < 1 || slices > MAX_SLICES || repeats < 1)
        return fail(AFQMC_OZAKI_ERR_ARG, "afqmc_ozaki_gemm: bad argument (1 <= slices <= 8, sizes >= 1)");
    if ((long long)K * 64 * 64 * slices >= (1LL << 31)) return fail(AFQMC_OZAKI_ERR_ARG, "afqmc_ozaki_gemm: K too large for exact INT32 accumulation");
    cudaStream_t stream = (cudaStream_t)stream_;
    int dev = 0, major = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (major != 10) return fail(AFQMC_OZAKI_ERR_ARCH, "afqmc_ozaki_gemm: needs sm_100");
    const int nk = (K + BK - 1) / BK, n_rt = (M + BM - 1) / BM, n_ct = (Ncol + BN - 1) / BN;
    const size_t a_sz = (size_t)n_rt * nk * slices * A_SLICE_BYTES, b_sz = (size_t)n_ct * nk * slices * B_SLICE_BYTES;
    int8_t *Ap = nullptr, *Bp = nullptr;
    double *sA = nullptr, *sB = nullptr, *csum = nullptr;
    int *err = nullptr;
    cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};
    int rc = AFQMC_OZAKI_OK;
    auto cleanup = [&]() {
        cudaFree(Ap); cudaFree(Bp); cudaFree(sA); cudaFree(sB); cudaFree(csum); cudaFree(err);
        for (auto &e : ev) if (e) cudaEventDestroy(e);
    };
#define OZ_TRY(call)                                                                                  \
    do {                                                                                              \
        cudaError_t e_ = (call);                                                                      \
        if (e_ != cudaSuccess) { g_err = std::string(#call) + ": " + cudaGetErrorString(e_); cleanup(); return AFQMC_OZAKI_ERR_CUDA; } \
    } while (0)
    OZ_TRY(cudaMalloc(&Ap, a_sz)); OZ_TRY(cudaMalloc(&Bp, b_sz));
    OZ_TRY(cudaMalloc(&sA, (size_t)M * 8)); OZ_TRY(cudaMalloc(&sB, (size_t)Ncol * 8));
    OZ_TRY(cudaMalloc(&csum, 8)); OZ_TRY(cudaMalloc(&err, 4));
    for (auto &e : ev) OZ_TRY(cudaEventCreate(&e));
    OZ_TRY(cudaMemsetAsync(Ap, 0, a_sz, stream)); OZ_TRY(cudaMemsetAsync(Bp, 0, b_sz, stream));
    OZ_TRY(cudaMemsetAsync(err, 0, 4, stream));
    const size_t smem = (size_t)STAGES * slices * (A_SLICE_BYTES + B_SLICE_BYTES) + 1024;
    OZ_TRY(cudaFuncSetAttribute((const void *)oz_gemm, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    OzParams p{};
    p.A = Ap; p.B = Bp; p.scaleA = sA; p.scaleB = sB; p.M = M; p.Ncol = Ncol; p.nk = nk; p.slices = slices; p.n_rt = n_rt; p.n_ct = n_ct;
    p.C = C; p.ldc = Ncol; p.checksum = csum; p.err = err;
    const int grid = (int)std::min<long long>((long long)n_rt * n_ct, sms);
    OZ_TRY(cudaEventRecord(ev[0], stream));
    for (int r = 0; r < repeats; ++r) {
        oz_slice<<<(M + 7) / 8, 256, 0, stream>>>(A, K, M, K, nk, slices, BM, Ap, sA);
        oz_slice<<<(Ncol + 7) / 8, 256, 0, stream>>>(B, K, Ncol, K, nk, slices, BN, Bp, sB);
    }
    OZ_TRY(cudaEventRecord(ev[1], stream));
    for (int r = 0; r < repeats; ++r) {
        OZ_TRY(cudaMemsetAsync(csum, 0, 8, stream));
        oz_gemm<<<grid, THREADS, smem, stream>>>(p);
    }
    OZ_TRY(cudaEventRecord(ev[2], stream));
    OZ_TRY(cudaGetLastError());
    OZ_TRY(cudaStreamSynchronize(stream));
    int herr = 0;
    OZ_TRY(cudaMemcpy(&herr, err, 4, cudaMemcpyDeviceToHost));
    if (herr != 0) {
        char buf[96];
        snprintf(buf, sizeof buf, "afqmc_ozaki_gemm: pipeline barrier %d timed out", herr);
        g_err = buf;
        rc = AFQMC_OZAKI_ERR_TIMEOUT;
    }
    float t = 0.f;
    if (ms_slice) { OZ_TRY(cudaEventElapsedTime(&t, ev[0], ev[1])); *ms_slice = t / repeats; }
    if (ms_gemm) { OZ_TRY(cudaEventElapsedTime(&t, ev[1], ev[2])); *ms_gemm = t / repeats; }
    if (checksum) OZ_TRY(cudaMemcpy(checksum, csum, 8, cudaMemcpyDeviceToHost));
#undef OZ_TRY
    cleanup();
    return rc;
}

}  // extern "C"
