/* A plain C99 client of include/afqmc.h (no Python, no C++): reads a problem from a binary file, evaluates the local
 * energies through the host-buffer entry point and through the device entry point, and writes both results.
 *
 *   afqmc_c_caller in.bin out.bin
 *   in.bin : int32 N, n_alpha, n_beta, n_gamma, n_walkers; float64 e0;
 *            float64 h1e[N*N], chol[n_gamma*N*N]; complex128 trial[N*(na+nb)], walkers[n_walkers*N*(na+nb)]
 *   out.bin: complex128 E_host[nw], logovlp_host[nw], E_dev[nw], logovlp_dev[nw]
 * Built and run by tests/test_c_caller.py; the layouts are those of the header.
 */
#include <stdio.h>
#include <stdlib.h>
#include <cuda_runtime_api.h>
#include "afqmc.h"

#define CHECK_CUDA(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { fprintf(stderr, "%s: %s\n", #x, cudaGetErrorString(e_)); return 2; } } while (0)

static void *slurp(FILE *f, size_t bytes) {
    void *p = malloc(bytes ? bytes : 1);
    if (!p || fread(p, 1, bytes, f) != bytes) { fprintf(stderr, "short read (%zu bytes)\n", bytes); exit(3); }
    return p;
}

int main(int argc, char **argv) {
    if (argc != 3) { fprintf(stderr, "usage: %s in.bin out.bin\n", argv[0]); return 1; }
    FILE *f = fopen(argv[1], "rb");
    if (!f) { perror(argv[1]); return 1; }
    int hdr[5];
    double e0;
    if (fread(hdr, sizeof(int), 5, f) != 5 || fread(&e0, sizeof(double), 1, f) != 1) { fprintf(stderr, "bad header\n"); return 3; }
    const int N = hdr[0], na = hdr[1], nb = hdr[2], ng = hdr[3], nw = hdr[4];
    const size_t h_bytes = (size_t)N * N * 8, c_bytes = (size_t)ng * N * N * 8, t_bytes = (size_t)N * (na + nb) * 16,
                 w_bytes = (size_t)nw * N * (na + nb) * 16, o_bytes = (size_t)nw * 16;
    double *h1e = slurp(f, h_bytes), *chol = slurp(f, c_bytes), *trial = slurp(f, t_bytes), *walkers = slurp(f, w_bytes);
    fclose(f);

    double *d_h1e, *d_chol, *d_trial, *d_walkers, *d_E, *d_O;
    CHECK_CUDA(cudaMalloc((void **)&d_h1e, h_bytes));
    CHECK_CUDA(cudaMalloc((void **)&d_chol, c_bytes));
    CHECK_CUDA(cudaMalloc((void **)&d_trial, t_bytes));
    CHECK_CUDA(cudaMalloc((void **)&d_walkers, w_bytes));
    CHECK_CUDA(cudaMalloc((void **)&d_E, o_bytes));
    CHECK_CUDA(cudaMalloc((void **)&d_O, o_bytes));
    CHECK_CUDA(cudaMemcpy(d_h1e, h1e, h_bytes, cudaMemcpyHostToDevice));
    CHECK_CUDA(cudaMemcpy(d_chol, chol, c_bytes, cudaMemcpyHostToDevice));
    CHECK_CUDA(cudaMemcpy(d_trial, trial, t_bytes, cudaMemcpyHostToDevice));
    CHECK_CUDA(cudaMemcpy(d_walkers, walkers, w_bytes, cudaMemcpyHostToDevice));

    afqmc_ctx *ctx = NULL;
    int rc = afqmc_create(d_h1e, d_chol, d_trial, N, na, nb, ng, e0, nw, NULL, &ctx);
    if (rc != AFQMC_OK) { fprintf(stderr, "afqmc_create: %d: %s\n", rc, afqmc_last_error(NULL)); return 4; }
    CHECK_CUDA(cudaFree(d_chol));                         /* "Not retained: may be freed after the call returns" */

    double *out = malloc(4 * o_bytes);
    rc = afqmc_local_energy_host(ctx, walkers, nw, out, out + 2 * (size_t)nw, NULL);
    if (rc != AFQMC_OK) { fprintf(stderr, "afqmc_local_energy_host: %d: %s\n", rc, afqmc_last_error(ctx)); return 4; }
    rc = afqmc_local_energy(ctx, d_walkers, nw, d_E, d_O, NULL);
    if (rc != AFQMC_OK) { fprintf(stderr, "afqmc_local_energy: %d: %s\n", rc, afqmc_last_error(ctx)); return 4; }
    CHECK_CUDA(cudaDeviceSynchronize());
    CHECK_CUDA(cudaMemcpy(out + 4 * (size_t)nw, d_E, o_bytes, cudaMemcpyDeviceToHost));
    CHECK_CUDA(cudaMemcpy(out + 6 * (size_t)nw, d_O, o_bytes, cudaMemcpyDeviceToHost));

    afqmc_info info;
    if (afqmc_get_info(ctx, &info) != AFQMC_OK || info.N != N || info.n_gamma != ng) { fprintf(stderr, "afqmc_get_info mismatch\n"); return 5; }
    /* argument errors are reported, not crashed on */
    if (afqmc_local_energy(ctx, d_walkers, nw + 1, d_E, d_O, NULL) != AFQMC_ERR_ARG) { fprintf(stderr, "n_walkers > max_walkers accepted\n"); return 5; }
    afqmc_destroy(ctx);

    f = fopen(argv[2], "wb");
    if (!f || fwrite(out, 1, 4 * o_bytes, f) != 4 * o_bytes) { perror(argv[2]); return 1; }
    fclose(f);
    printf("afqmc_c_caller: %d walkers, N=%d, E[0] = %.12g %+.12gi, kernel launches %lld\n", nw, N, out[0], out[1], info.kernel_launches);
    return 0;
}
