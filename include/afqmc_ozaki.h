/*
 * afqmc_ozaki.h -- C ABI of the Ozaki-scheme EXPERIMENT: FP64 emulation of the contraction
 *     T^gamma = Ltilde^gamma theta^T                                              PAPER.md:237-242 (Eq. 29)
 * as a real GEMM  C[M x Ncol] = A[M x K] B[Ncol x K]^T  on the INT8 tensor cores (tcgen05.mma kind::i8, TMEM
 * accumulators), built as its own library (libafqmc_ozaki.so).  It is NOT on the product path of include/afqmc.h;
 * profiles/r2_ozaki.md has the measured accuracy / throughput and the go / no-go.
 *
 * Scheme (csrc/ozaki_i8.cu): every row of A and of B is scaled by a power of two and cut into `slices` signed 7-bit
 * digits (exact in FP64); the slices (slices + 1) / 2 integer products A_s B_t^T with s + t < slices are exact in
 * INT32, products of equal weight s + t share one TMEM accumulator, and the epilogue recombines them in FP64.
 * Relative truncation ~ K 2^(-7 slices) against max_k|a_ik| max_k|b_jk|.
 */
#ifndef AFQMC_OZAKI_H_
#define AFQMC_OZAKI_H_

#ifdef __cplusplus
extern "C" {
#endif

enum {
    AFQMC_OZAKI_OK = 0,
    AFQMC_OZAKI_ERR_ARG = -1,
    AFQMC_OZAKI_ERR_CUDA = -3,
    AFQMC_OZAKI_ERR_ARCH = -4,
    AFQMC_OZAKI_ERR_TIMEOUT = -6 /* a pipeline barrier of the kernel did not complete (bounded waits; the kernel exits) */
};

/*
 * afqmc_ozaki_gemm -- C = A B^T through `slices` INT8 digit planes.
 *   A         device, float64 [M][K] row-major   (rows of Ltilde: (gamma, i), K = N orbitals)
 *   B         device, float64 [Ncol][K] row-major (rows = columns of C: (plane, walker, j) of theta)
 *   slices    1 .. 8
 *   C         device, float64 [M][Ncol] row-major, or NULL: nothing is stored (timing runs at sizes whose C would not fit)
 *   checksum  host, or NULL: sum over all elements of C^2 (accumulated with atomics: not bit-reproducible)
 *   ms_slice  host, or NULL: device time of cutting A and B into digits, per repeat
 *   ms_gemm   host, or NULL: device time of the tcgen05 kernel (products + FP64 recombination), per repeat
 *   repeats   >= 1: slicing and kernel are each run this many times back to back for the timings
 * Allocates and frees its own workspaces, synchronises `stream` before returning.
 */
int afqmc_ozaki_gemm(const double *A, const double *B, int M, int Ncol, int K, int slices, double *C, double *checksum,
                     float *ms_slice, float *ms_gemm, int repeats, void *stream);

/* Message of the last error on this thread. */
const char *afqmc_ozaki_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* AFQMC_OZAKI_H_ */
