// Shared device helpers and the packed-operand layout used by K0 (setup), K1 (theta) and K2 (exchange).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace afqmc {

// ------------------------------------------------------------------------------------------------
// Packed operand layout ("fragment order").
//
// K2 computes, per spin, the real TN product  C[(gamma,i)][(plane,w,j)] = sum_p Lt[gamma][i][p] * theta[w][j][p][plane]
// (Eq. 29, with the real/imag split of PAPER.md:212, 260-268) with DMMA.8x8x4.  One m8n8k4
// A fragment is an 8-row x 4-k block with lane l holding (row l/4, k l%4); the col-major B fragment is the same
// with "row" = output column.  Both operands are library-owned, so they are stored directly as those 32-double
// blocks:
//
//      operand[tile][kstep][strip][lane]      strip = 8 consecutive rows (cols) of the CTA tile, lane = r*4 + k
//
// A CTA tile of the A operand holds g_tile whole gamma-blocks (g_tile*n rows, zero-padded up to R = 8*strips);
// a CTA tile of the B operand holds both planes of w_tile walkers, column = (plane*w_tile + wl)*n + j,
// zero-padded up to C.  k is zero-padded from N to 4*ksteps.  A K-chunk (consecutive ksteps) of a tile is one
// contiguous block, fetched with a single 1-D bulk async copy, and every fragment load from shared memory is
// 256 contiguous bytes (bank-conflict free).
// ------------------------------------------------------------------------------------------------
struct OperandLayout {
    int n;          // electrons of this spin
    int strips;     // 8-row strips per tile (R/8 or C/8)
    int ksteps;     // ceil(N/4)
    int per_tile;   // gamma-blocks (A) or walkers (B) per tile
    long long tile_doubles;  // strips * ksteps * 32
};

__host__ __device__ inline long long packed_offset(const OperandLayout &L, int tile, int row_in_tile, int p) {
    int s = row_in_tile >> 3, rr = row_in_tile & 7, ks = p >> 2, kk = p & 3;
    return (long long)tile * L.tile_doubles + ((long long)ks * L.strips + s) * 32 + rr * 4 + kk;
}

// ------------------------------------------------------------------------------------------------
// PTX wrappers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void dmma_m8n8k4(double &d0, double &d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra.uni WAIT_DONE;\n"
        "bra.uni WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// 1-D bulk async copy global -> shared, completion counted in bytes on an mbarrier (TMA engine, UBLKCP in SASS).
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;\n" ::"r"(id), "r"(nthreads) : "memory");
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

}  // namespace afqmc
