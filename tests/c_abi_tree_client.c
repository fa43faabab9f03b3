/*
 * c_abi_tree_client.c -- a plain C program that runs the adaptive-tree solve through include/octo_fmm.h only (no Python, no
 * torch): octo_fmm_tree_workspace_bytes / create / interaction_counts (= solve + pair counts) / status / destroy, with device
 * memory from the CUDA runtime.  tests/test_gpu_c_abi.py builds it with nvcc, runs it and compares the output with the oracle.
 *
 * input file : int32 n0, depth, correction; double h0, theta; int32 box[depth][6]; then per level kind (uint8, box cells)
 *              and mass (double, box cells)
 * output file: per level out [4][box cells] (double); then uint64 counts[3]
 */
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

#include "octo_fmm.h"

#define CHECK(cond, msg) do { if (!(cond)) { fprintf(stderr, "c_abi_tree_client: %s\n", msg); return 1; } } while (0)
#define MAXD 12

int main(int argc, char **argv)
{
    CHECK(argc == 3, "usage: c_abi_tree_client <input> <output>");
    FILE *f = fopen(argv[1], "rb");
    CHECK(f, "cannot open input");
    int32_t hdr[3];
    double hd[2];
    CHECK(fread(hdr, sizeof(int32_t), 3, f) == 3 && fread(hd, sizeof(double), 2, f) == 2, "short header");
    const int depth = hdr[1];
    CHECK(depth >= 1 && depth <= MAXD, "bad depth");
    int box[MAXD * 6];
    CHECK(fread(box, sizeof(int32_t), (size_t)6 * depth, f) == (size_t)6 * depth, "short boxes");
    unsigned char *kind[MAXD];
    double *mass_h[MAXD], *mass_d[MAXD], *out_d[MAXD];
    size_t cells[MAXD];
    for (int l = 0; l < depth; ++l) {
        cells[l] = (size_t)box[6 * l + 3] * box[6 * l + 4] * box[6 * l + 5];
        kind[l] = (unsigned char *)malloc(cells[l]);
        mass_h[l] = (double *)malloc(cells[l] * sizeof(double));
        CHECK(kind[l] && mass_h[l], "out of host memory");
        CHECK(fread(kind[l], 1, cells[l], f) == cells[l] && fread(mass_h[l], sizeof(double), cells[l], f) == cells[l], "short level");
    }
    fclose(f);

    octo_fmm_tree_config cfg = {0};
    cfg.n0 = hdr[0];
    cfg.depth = depth;
    cfg.h0 = hd[0];
    cfg.theta = hd[1];
    cfg.am_correction = hdr[2];
    cfg.device = 0;
    cudaStream_t stream;
    CHECK(cudaSetDevice(0) == cudaSuccess && cudaStreamCreate(&stream) == cudaSuccess, "no CUDA device");
    cfg.stream = stream;
    cfg.workspace_bytes = octo_fmm_tree_workspace_bytes(&cfg, (const unsigned char *const *)kind, box);
    CHECK(cfg.workspace_bytes > 0, "configuration refused");
    CHECK(cudaMalloc(&cfg.workspace, cfg.workspace_bytes) == cudaSuccess, "cudaMalloc workspace");
    for (int l = 0; l < depth; ++l) {
        CHECK(cudaMalloc((void **)&mass_d[l], cells[l] * sizeof(double)) == cudaSuccess &&
              cudaMalloc((void **)&out_d[l], 4 * cells[l] * sizeof(double)) == cudaSuccess, "cudaMalloc level");
        CHECK(cudaMemcpyAsync(mass_d[l], mass_h[l], cells[l] * sizeof(double), cudaMemcpyHostToDevice, stream) == cudaSuccess, "H2D");
    }
    octo_fmm_tree_t *t = NULL;
    CHECK(octo_fmm_tree_create(&cfg, (const unsigned char *const *)kind, box, &t) == OCTO_FMM_OK, "octo_fmm_tree_create");
    unsigned long long counts[3] = {0, 0, 0};
    CHECK(octo_fmm_tree_interaction_counts(t, (const double *const *)mass_d, out_d, counts) == OCTO_FMM_OK, "octo_fmm_tree_interaction_counts");
    CHECK(octo_fmm_tree_solve(t, (const double *const *)mass_d, out_d) == OCTO_FMM_OK, "octo_fmm_tree_solve");     /* a plain solve on top */
    CHECK(octo_fmm_tree_status(t) == OCTO_FMM_OK, "octo_fmm_tree_status");
    int launches = 0;
    CHECK(octo_fmm_tree_launches(t, &launches) == OCTO_FMM_OK && launches > 0, "octo_fmm_tree_launches");

    FILE *g = fopen(argv[2], "wb");
    CHECK(g, "cannot open output");
    for (int l = 0; l < depth; ++l) {
        double *o = (double *)malloc(4 * cells[l] * sizeof(double));
        CHECK(o, "out of host memory");
        CHECK(cudaMemcpy(o, out_d[l], 4 * cells[l] * sizeof(double), cudaMemcpyDeviceToHost) == cudaSuccess, "D2H");
        CHECK(fwrite(o, sizeof(double), 4 * cells[l], g) == 4 * cells[l], "short write");
        free(o);
    }
    uint64_t c64[3] = {counts[0], counts[1], counts[2]};
    CHECK(fwrite(c64, sizeof(uint64_t), 3, g) == 3, "short write");
    fclose(g);
    CHECK(octo_fmm_tree_destroy(t) == OCTO_FMM_OK, "octo_fmm_tree_destroy");
    for (int l = 0; l < depth; ++l) { cudaFree(mass_d[l]); cudaFree(out_d[l]); free(kind[l]); free(mass_h[l]); }
    cudaFree(cfg.workspace);
    cudaStreamDestroy(stream);
    return 0;
}
