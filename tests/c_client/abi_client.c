/* A plain C client of the C ABI (include/gdrr.h): no Python, no torch -- only the CUDA runtime for device memory.
 * tests/test_gpu_c_client.py compiles it with gcc, runs it on the GPU and compares what it prints with the oracle.
 *
 *   abi_client <libgdrr_b200.so is linked> : builds a 24 x 20 x 16 volume of two materials from a closed formula,
 *   projects three gantry angles of a 40 x 30 detector with a 3-bin spectrum and prints every signal value.
 */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>

#include <cuda_runtime.h>

#include "gdrr.h"

#define CHECK_CUDA(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { fprintf(stderr, "CUDA: %s\n", cudaGetErrorString(e_)); return 2; } } while (0)
#define CHECK_GDRR(x) do { int r_ = (x); if (r_ != GDRR_OK) { fprintf(stderr, "gdrr error %d: %s\n", r_, gdrr_last_error(ctx)); return 3; } } while (0)

int main(void) {
    enum { NX = 24, NY = 20, NZ = 16, NU = 40, NV = 30, NP = 3, NE = 3, NM = 2 };
    static float rho[NZ][NY][NX];
    static unsigned char mat[NZ][NY][NX];
    for (int z = 0; z < NZ; ++z)
        for (int y = 0; y < NY; ++y)
            for (int x = 0; x < NX; ++x) {
                /* the same formula is in tests/test_gpu_c_client.py */
                rho[z][y][x] = 0.25f * (float)((x * 7 + y * 3 + z * 5) % 9);
                mat[z][y][x] = (unsigned char)((x + 2 * y + 3 * z) % 7 < 3 ? 1 : 0);
            }
    const double phi[NP] = {0.0, 0.7, 3.3};
    const double phi_weight[NE] = {0.2, 0.5, 0.3}, response[NE] = {0.6, 1.0, 1.4};
    const double mu_hat[NM][NE] = {{0.030, 0.022, 0.018}, {0.060, 0.035, 0.025}};

    gdrr_context* ctx = NULL;
    if (gdrr_create_context(0, &ctx) != GDRR_OK) { fprintf(stderr, "%s\n", gdrr_last_error(NULL)); return 1; }
    CHECK_GDRR(gdrr_set_geometry(ctx, 1000.0, 1500.0, 0.0, NU, NV, 1.2, 1.2, 0.0, 0.0, NP, phi, 0.6));
    CHECK_GDRR(gdrr_set_spectrum(ctx, NE, NM, phi_weight, response, &mu_hat[0][0], NULL, NULL, NULL));

    float *rho_dev = NULL, *signal_dev = NULL;
    unsigned char* mat_dev = NULL;
    void* ws = NULL;
    size_t ws_bytes = 0;
    CHECK_GDRR(gdrr_volume_workspace_bytes(NX, NY, NZ, NM, GDRR_LAYOUT_PACKED_QUAD, &ws_bytes));
    CHECK_CUDA(cudaMalloc((void**)&rho_dev, sizeof rho));
    CHECK_CUDA(cudaMalloc((void**)&mat_dev, sizeof mat));
    CHECK_CUDA(cudaMalloc(&ws, ws_bytes));
    CHECK_CUDA(cudaMalloc((void**)&signal_dev, sizeof(float) * NP * NV * NU));
    CHECK_CUDA(cudaMemcpy(rho_dev, rho, sizeof rho, cudaMemcpyHostToDevice));
    CHECK_CUDA(cudaMemcpy(mat_dev, mat, sizeof mat, cudaMemcpyHostToDevice));

    gdrr_volume* vol = NULL;
    CHECK_GDRR(gdrr_create_volume(ctx, rho_dev, mat_dev, NX, NY, NZ, 1.5, 1.5, 2.0, NULL, NM, GDRR_LAYOUT_PACKED_QUAD,
                                  ws, ws_bytes, NULL, &vol));
    CHECK_GDRR(gdrr_volume_status(ctx, vol));
    CHECK_GDRR(gdrr_project(ctx, vol, 0, NP, signal_dev, NULL, NULL, NULL));
    CHECK_CUDA(cudaDeviceSynchronize());

    static float signal[NP][NV][NU];
    CHECK_CUDA(cudaMemcpy(signal, signal_dev, sizeof signal, cudaMemcpyDeviceToHost));
    printf("launches %llu sampler %d version %s\n", gdrr_kernel_launches(ctx), gdrr_last_sampler(ctx), gdrr_version());
    for (int p = 0; p < NP; ++p)
        for (int j = 0; j < NV; ++j)
            for (int i = 0; i < NU; ++i) printf("%.9g\n", signal[p][j][i]);

    /* the host-buffer entry points give the same bits */
    static float signal_h[NP][NV][NU];
    gdrr_volume* vol_h = NULL;
    CHECK_GDRR(gdrr_create_volume_host(ctx, &rho[0][0][0], &mat[0][0][0], NX, NY, NZ, 1.5, 1.5, 2.0, NULL, NM,
                                       GDRR_LAYOUT_PACKED_QUAD, rho_dev, mat_dev, ws, ws_bytes, NULL, &vol_h));
    CHECK_GDRR(gdrr_project_host(ctx, vol_h, 0, NP, &signal_h[0][0][0], signal_dev, NP, NULL));
    int same = 1;
    for (int k = 0; k < NP * NV * NU; ++k) same = same && (&signal[0][0][0])[k] == (&signal_h[0][0][0])[k];
    printf("host path identical %d\n", same);

    gdrr_destroy_volume(vol_h);
    gdrr_destroy_volume(vol);
    gdrr_destroy_context(ctx);
    cudaFree(rho_dev); cudaFree(mat_dev); cudaFree(ws); cudaFree(signal_dev);
    return 0;
}
