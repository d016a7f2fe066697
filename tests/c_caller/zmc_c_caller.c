/* A plain C99 caller of the C ABI (include/zmc.h): no Python, no torch.  Test infrastructure: built and run by
 * tests/test_gpu_c_caller.py, which compares what it writes with the CPU oracle.
 * Scans cfg 1's family (g = cos(x1 y), y in [0,1]) over argv[2] linspace values of x1 in [0.1, 10] with argv[3] samples:
 * once through zmc_scan into device memory (copied back here) and once through zmc_scan_ex into HOST memory in batches
 * of 7 points; writes mean[], stderr[] of the first scan and then of the second as raw doubles to argv[1]. */
#include <stdio.h>
#include <stdlib.h>
#include <cuda_runtime_api.h>
#include "zmc.h"

int main(int argc, char** argv)
{
    if (argc != 4) return 2;
    const int L = atoi(argv[2]);
    const uint64_t n = (uint64_t)atoll(argv[3]);
    double* x = (double*)malloc(sizeof(double) * (size_t)L);
    for (int j = 0; j < L; ++j) x[j] = 0.1 + j * ((10.0 - 0.1) / (L - 1));
    x[L - 1] = 10.0;
    const double bounds[2] = {0.0, 1.0};
    zmc_param_list list = {x, L};

    double *d_mean = NULL, *d_err = NULL;
    if (cudaMalloc((void**)&d_mean, sizeof(double) * L) != cudaSuccess || cudaMalloc((void**)&d_err, sizeof(double) * L) != cudaSuccess) return 3;
    cudaStream_t stream;
    if (cudaStreamCreate(&stream) != cudaSuccess) return 3;
    zmc_status st = zmc_scan(ZMC_FAM_C1_COS_XY, 1, bounds, 1, &list, n, 1, d_mean, d_err, (void*)stream);
    if (st != ZMC_OK) { fprintf(stderr, "zmc_scan: %s\n", zmc_status_string(st)); return 4; }
    double* h = (double*)malloc(sizeof(double) * 4 * (size_t)L);
    if (cudaMemcpyAsync(h, d_mean, sizeof(double) * L, cudaMemcpyDeviceToHost, stream) != cudaSuccess) return 3;
    if (cudaMemcpyAsync(h + L, d_err, sizeof(double) * L, cudaMemcpyDeviceToHost, stream) != cudaSuccess) return 3;

    zmc_options o = {0};
    o.struct_size = sizeof(o);
    o.out_location = ZMC_LOC_HOST;
    o.batch_points = 7;
    double *p_mean = NULL, *p_err = NULL;                      /* page-locked, as the header recommends */
    if (cudaMallocHost((void**)&p_mean, sizeof(double) * L) != cudaSuccess || cudaMallocHost((void**)&p_err, sizeof(double) * L) != cudaSuccess) return 3;
    zmc_timing tm;
    st = zmc_scan_ex(ZMC_FAM_C1_COS_XY, 1, bounds, 1, &list, n, 1, p_mean, p_err, (void*)stream, &o, &tm);
    if (st != ZMC_OK) { fprintf(stderr, "zmc_scan_ex: %s\n", zmc_status_string(st)); return 4; }
    if (cudaStreamSynchronize(stream) != cudaSuccess) return 3;
    if (tm.n_batches != (L + 6) / 7 || tm.host_out_pinned != 1) { fprintf(stderr, "timing: %lld batches, pinned %d\n", (long long)tm.n_batches, tm.host_out_pinned); return 5; }
    for (int j = 0; j < L; ++j) { h[2 * L + j] = p_mean[j]; h[3 * L + j] = p_err[j]; }

    /* an argument error returns before anything is enqueued */
    if (zmc_scan(ZMC_FAM_C1_COS_XY, 2, bounds, 1, &list, n, 1, d_mean, d_err, (void*)stream) == ZMC_OK) return 6;

    FILE* f = fopen(argv[1], "wb");
    if (!f || fwrite(h, sizeof(double), 4 * (size_t)L, f) != 4 * (size_t)L) return 7;
    fclose(f);
    zmc_shutdown();
    printf("%s ok\n", zmc_version());
    return 0;
}
