/*
 * c_abi_client.c -- a plain C program that uses the library through include/octo_fmm.h only (no Python, no torch):
 * it reads a seeded workload from a file, allocates device memory with the CUDA runtime, runs
 * create / set_moments / interact / get_expansions / destroy and writes the expansions to a file.
 * tests/test_gpu_c_abi.py builds it with nvcc, runs it and compares the output with the oracle.
 *
 * input file : int32 n[3], out_lo[3], out_hi[3], correction; double h, theta; then moments [20][nz][ny][nx], com_off [3][..]
 * output file: double L [20][out cells], Lcorr [3][out cells]; uint64 interaction count; int32 stencil count of class 0
 */
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

#include "octo_fmm.h"

#define CHECK(cond, msg) do { if (!(cond)) { fprintf(stderr, "c_abi_client: %s\n", msg); return 1; } } while (0)

int main(int argc, char **argv)
{
    CHECK(argc == 3, "usage: c_abi_client <input> <output>");
    FILE *f = fopen(argv[1], "rb");
    CHECK(f, "cannot open input");
    int32_t hdr[10];
    double hd[2];
    CHECK(fread(hdr, sizeof(int32_t), 10, f) == 10 && fread(hd, sizeof(double), 2, f) == 2, "short header");
    const size_t ncell = (size_t)hdr[0] * hdr[1] * hdr[2];
    const size_t ocell = (size_t)(hdr[6] - hdr[3]) * (hdr[7] - hdr[4]) * (hdr[8] - hdr[5]);
    double *mom = (double *)malloc(ncell * 20 * sizeof(double)), *com = (double *)malloc(ncell * 3 * sizeof(double));
    CHECK(mom && com, "out of host memory");
    CHECK(fread(mom, sizeof(double), ncell * 20, f) == ncell * 20 && fread(com, sizeof(double), ncell * 3, f) == ncell * 3,
          "short payload");
    fclose(f);

    octo_fmm_config cfg = {0};
    for (int a = 0; a < 3; ++a) { cfg.n[a] = hdr[a]; cfg.out_lo[a] = hdr[3 + a]; cfg.out_hi[a] = hdr[6 + a]; }
    cfg.h = hd[0];
    cfg.theta = hd[1];
    cfg.kind = OCTO_FMM_MULTIPOLE;
    cfg.am_correction = hdr[9];
    cfg.device = 0;
    cudaStream_t stream;
    CHECK(cudaStreamCreate(&stream) == cudaSuccess, "no CUDA device");
    cfg.stream = stream;
    cfg.workspace_bytes = octo_fmm_workspace_bytes(&cfg);
    CHECK(cfg.workspace_bytes > 0, "configuration rejected");
    double *d_mom, *d_com, *d_L, *d_C;
    CHECK(cudaMalloc(&cfg.workspace, cfg.workspace_bytes) == cudaSuccess && cudaMalloc((void **)&d_mom, ncell * 20 * 8) == cudaSuccess &&
          cudaMalloc((void **)&d_com, ncell * 3 * 8) == cudaSuccess && cudaMalloc((void **)&d_L, ocell * 20 * 8) == cudaSuccess &&
          cudaMalloc((void **)&d_C, ocell * 3 * 8) == cudaSuccess, "cudaMalloc failed");
    CHECK(cudaMemcpyAsync(d_mom, mom, ncell * 20 * 8, cudaMemcpyHostToDevice, stream) == cudaSuccess, "H2D");
    CHECK(cudaMemcpyAsync(d_com, com, ncell * 3 * 8, cudaMemcpyHostToDevice, stream) == cudaSuccess, "H2D");

    octo_fmm_t *h = NULL;
    CHECK(octo_fmm_interact(NULL) == OCTO_FMM_EINVAL, "NULL handle must be EINVAL");
    CHECK(octo_fmm_create(&cfg, &h) == OCTO_FMM_OK, "create");
    CHECK(octo_fmm_interact(h) == OCTO_FMM_ESTATE, "interact before set_moments must be ESTATE");
    CHECK(octo_fmm_set_moments(h, d_mom, d_com) == OCTO_FMM_OK, "set_moments");
    CHECK(octo_fmm_get_expansions(h, d_L, d_C) == OCTO_FMM_ESTATE, "get before interact must be ESTATE");
    CHECK(octo_fmm_interact(h) == OCTO_FMM_OK, "interact");
    CHECK(octo_fmm_get_expansions(h, d_L, d_C) == OCTO_FMM_OK, "get_expansions");
    CHECK(octo_fmm_status(h) == OCTO_FMM_OK, "status");
    unsigned long long count = 0;
    int32_t nst = 0;
    CHECK(octo_fmm_interaction_count(h, &count) == OCTO_FMM_OK, "interaction_count");
    CHECK(octo_fmm_get_stencil(h, 0, &nst, NULL) == OCTO_FMM_OK, "get_stencil");

    double *L = (double *)malloc(ocell * 23 * sizeof(double));
    CHECK(L, "out of host memory");
    CHECK(cudaMemcpy(L, d_L, ocell * 20 * 8, cudaMemcpyDeviceToHost) == cudaSuccess, "D2H");
    CHECK(cudaMemcpy(L + ocell * 20, d_C, ocell * 3 * 8, cudaMemcpyDeviceToHost) == cudaSuccess, "D2H");
    CHECK(octo_fmm_destroy(h) == OCTO_FMM_OK, "destroy");

    f = fopen(argv[2], "wb");
    CHECK(f, "cannot open output");
    uint64_t c64 = count;
    CHECK(fwrite(L, sizeof(double), ocell * 23, f) == ocell * 23 && fwrite(&c64, sizeof c64, 1, f) == 1 &&
          fwrite(&nst, sizeof nst, 1, f) == 1, "short write");
    fclose(f);
    printf("c_abi_client: %s, %llu interactions\n", octo_fmm_version(), count);
    return 0;
}
