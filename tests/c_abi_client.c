/* c_abi_client.c -- libdebye called from plain C: no Python, no torch, only include/debye.h and the CUDA runtime for the
 * caller's own buffers.  Built and run by tests/test_parity_gpu.py::test_c_abi_from_plain_c, which writes the input file,
 * compares the profiles this program writes with the oracle and prints the latencies it measures.
 *
 *   c_abi_client <in.bin> <out.bin> <repetitions>
 *   in.bin : int32 N, T, M; float xyz[N][3]; int32 type[N]; float fftab[T][M]; float q[M]
 *   out.bin: double I_host[M] (debye_profile_host, host buffers); double I_dev[M] (debye_profile, device buffers);
 *            double I_static[M] (debye_profile_static, or NaN if the input is beyond its limits);
 *            double us_host, us_dev_sync, us_dev_back_to_back  (microseconds per call)
 */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <time.h>
#include <cuda_runtime.h>
#include "debye.h"

static double now(void) { struct timespec t; clock_gettime(CLOCK_MONOTONIC, &t); return t.tv_sec + 1e-9 * t.tv_nsec; }
#define CHECK(call)                                                                         \
    do {                                                                                    \
        int st__ = (call);                                                                  \
        if (st__ != 0) { fprintf(stderr, "%s -> %d (%s)\n", #call, st__, debye_strerror(st__)); return 2; } \
    } while (0)
#define CUDA(call)                                                                          \
    do {                                                                                    \
        cudaError_t e__ = (call);                                                           \
        if (e__ != cudaSuccess) { fprintf(stderr, "%s -> %s\n", #call, cudaGetErrorString(e__)); return 3; } \
    } while (0)

int main(int argc, char **argv)
{
    if (argc < 4) { fprintf(stderr, "usage: %s in.bin out.bin repetitions\n", argv[0]); return 1; }
    FILE *fi = fopen(argv[1], "rb");
    if (!fi) { perror(argv[1]); return 1; }
    const int reps = atoi(argv[3]);
    int32_t hdr[3];
    if (fread(hdr, 4, 3, fi) != 3) return 1;
    const int N = hdr[0], T = hdr[1], M = hdr[2];
    float *xyz, *f, *q;
    int32_t *type;
    double *out;
    /* pinned host buffers (pageable ones work too: the library stages small inputs itself) */
    CUDA(cudaHostAlloc((void **)&xyz, (size_t)N * 12, 0));
    CUDA(cudaHostAlloc((void **)&type, (size_t)N * 4, 0));
    CUDA(cudaHostAlloc((void **)&f, (size_t)T * M * 4, 0));
    CUDA(cudaHostAlloc((void **)&q, (size_t)M * 4, 0));
    CUDA(cudaHostAlloc((void **)&out, (size_t)M * 8 * 3, 0));
    if (fread(xyz, 12, N, fi) != (size_t)N || fread(type, 4, N, fi) != (size_t)N || fread(f, 4, (size_t)T * M, fi) != (size_t)T * M ||
        fread(q, 4, M, fi) != (size_t)M)
        return 1;
    fclose(fi);
    double *I_host = out, *I_dev = out + M, *I_static = out + 2 * M;
    const uint32_t hint = debye_q_hint(q, M);       /* the grid is known on the host: one pairs launch (one launch in all if small) */
    cudaStream_t s;
    CUDA(cudaStreamCreate(&s));

    /* 1. host buffers in, host buffer out */
    for (int i = 0; i < 10; ++i) CHECK(debye_profile_host(xyz, type, N, f, T, q, M, I_host, hint, (debye_stream_t)s));
    double t0 = now();
    for (int i = 0; i < reps; ++i) CHECK(debye_profile_host(xyz, type, N, f, T, q, M, I_host, hint, (debye_stream_t)s));
    const double us_host = (now() - t0) / reps * 1e6;

    /* 2. the caller's own device buffers */
    float *dx, *df, *dq;
    int32_t *dt;
    double *dout;
    CUDA(cudaMalloc((void **)&dx, (size_t)N * 12));
    CUDA(cudaMalloc((void **)&dt, (size_t)N * 4));
    CUDA(cudaMalloc((void **)&df, (size_t)T * M * 4));
    CUDA(cudaMalloc((void **)&dq, (size_t)M * 4));
    CUDA(cudaMalloc((void **)&dout, (size_t)M * 8));
    CUDA(cudaMemcpy(dx, xyz, (size_t)N * 12, cudaMemcpyHostToDevice));
    CUDA(cudaMemcpy(dt, type, (size_t)N * 4, cudaMemcpyHostToDevice));
    CUDA(cudaMemcpy(df, f, (size_t)T * M * 4, cudaMemcpyHostToDevice));
    CUDA(cudaMemcpy(dq, q, (size_t)M * 4, cudaMemcpyHostToDevice));
    for (int i = 0; i < 10; ++i) CHECK(debye_profile(dx, dt, N, df, T, dq, M, dout, hint, (debye_stream_t)s));
    CUDA(cudaStreamSynchronize(s));
    t0 = now();
    for (int i = 0; i < reps; ++i) {
        CHECK(debye_profile(dx, dt, N, df, T, dq, M, dout, hint, (debye_stream_t)s));
        CUDA(cudaStreamSynchronize(s));
    }
    const double us_sync = (now() - t0) / reps * 1e6;
    t0 = now();
    for (int i = 0; i < reps; ++i) CHECK(debye_profile(dx, dt, N, df, T, dq, M, dout, hint, (debye_stream_t)s));
    CUDA(cudaStreamSynchronize(s));
    const double us_b2b = (now() - t0) / reps * 1e6;
    CUDA(cudaMemcpy(I_dev, dout, (size_t)M * 8, cudaMemcpyDeviceToHost));

    /* 3. the entry that allocates nothing (small structures on hinted uniform grids only) */
    CUDA(cudaMemset(dout, 0xff, (size_t)M * 8));
    int st = debye_profile_static(dx, dt, N, df, T, dq, M, dout, hint, (debye_stream_t)s);
    if (st == DEBYE_OK) {
        CUDA(cudaStreamSynchronize(s));
        CUDA(cudaMemcpy(I_static, dout, (size_t)M * 8, cudaMemcpyDeviceToHost));
    } else {
        fprintf(stderr, "debye_profile_static: %s\n", debye_profile_static_error());
        for (int k = 0; k < M; ++k) I_static[k] = NAN;
    }

    FILE *fo = fopen(argv[2], "wb");
    if (!fo) { perror(argv[2]); return 1; }
    const double lat[3] = {us_host, us_sync, us_b2b};
    fwrite(out, 8, (size_t)3 * M, fo);
    fwrite(lat, 8, 3, fo);
    fclose(fo);
    printf("N = %d, T = %d, M = %d: debye_profile_host %.1f us per call; debye_profile + synchronise %.1f us; debye_profile back to back %.1f us\n",
           N, T, M, us_host, us_sync, us_b2b);
    debye_shutdown();
    return 0;
}
