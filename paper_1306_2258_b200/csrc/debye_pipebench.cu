// debye_pipebench.cu -- diagnostic micro-kernels behind debye_pipe_bench() (include/debye.h): what one SM of this part
// delivers on the instruction mixes the pairs kernels are made of, and the error statistics of MUFU.SIN.  These are the
// measured denominators / side conditions of the "alu" roofline ("these are nominal; the build must
// measure them"); bench.py --peaks prints them, profiles/ keeps the output.  Not on the hot path.
#include <cuda_runtime.h>
#include <cstdint>
#include <cmath>
#include "../../include/debye.h"
#include "debye_pairs.cuh"

namespace {
using namespace debye;

// every test: `iters` trips of an unrolled body; per warp the SM cycle counter (clock64) at start and end and the SM id
// the lane-operations and instructions per trip are in the host table below
template <int TEST>
__global__ void __launch_bounds__(128) pipe_kernel(int iters, const float *__restrict__ init, long long *__restrict__ cycles, float *__restrict__ sink)
{
    const int tid = threadIdx.x;
    // operands come from memory so that the compiler knows no relation between them
    float a = init[0], b = init[1];
    float x[16];
    u64 p[16], q2[4];
#pragma unroll
    for (int i = 0; i < 16; ++i) { x[i] = init[2 + i]; p[i] = pk2(init[18 + i], init[34 + i]); }
#pragma unroll
    for (int i = 0; i < 4; ++i) q2[i] = pk2(init[50 + i], init[54 + i]);
    const u64 a2 = pk2(a, a);
    u64 acc[56];
#pragma unroll
    for (int i = 0; i < 56; ++i) acc[i] = pk2(0.f, 0.f);
    unsigned iv = tid;
    __syncthreads();
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
        if constexpr (TEST == 0) {            // scalar FFMA, 16 independent chains x 4
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int i = 0; i < 16; ++i) x[i] = fmaf(x[i], a, b);
        } else if constexpr (TEST == 1) {     // FFMA2, 16 independent chains x 4, multiplier in scalar-broadcast form
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int i = 0; i < 16; ++i) p[i] = fma2(a2, p[i], q2[i & 3]);
        } else if constexpr (TEST == 2) {     // FADD2, 16 chains x 4
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int i = 0; i < 16; ++i) p[i] = add2(p[i], q2[i & 3]);
        } else if constexpr (TEST == 3) {     // the product form's outer product: 14 weights x 4 seed pairs, 56 accumulators
#pragma unroll
            for (int j = 0; j < 14; ++j) {
                const u64 w = pk2(x[j], x[j]);
#pragma unroll
                for (int c = 0; c < 4; ++c) acc[4 * j + c] = fma2(w, q2[c], acc[4 * j + c]);
            }
        } else if constexpr (TEST == 4) {     // the chain form's step: FADD2 accumulate + FFMA2 advance, 4 chains, 14 steps
#pragma unroll
            for (int j = 0; j < 14; ++j)
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    acc[4 * j + c] = add2(acc[4 * j + c], p[c]);
                    const u64 nx = fma2(a2, p[c], p[4 + c]);
                    p[4 + c] = p[c]; p[c] = nx;
                }
        } else if constexpr (TEST == 5) {     // MUFU.SIN, 16 chains x 2 (sin.approx = FMUL.RZ + MUFU.SIN)
#pragma unroll
            for (int r = 0; r < 2; ++r)
#pragma unroll
                for (int i = 0; i < 16; ++i) x[i] = sin_mufu(x[i]);
        } else if constexpr (TEST == 6) {     // outer product with one ALU-pipe instruction (LOP3) per FFMA2
#pragma unroll
            for (int j = 0; j < 14; ++j) {
                const u64 w = pk2(x[j], x[j]);
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    acc[4 * j + c] = fma2(w, q2[c], acc[4 * j + c]);
                    asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(iv) : "r"(it), "r"(tid + c));
                }
            }
        } else if constexpr (TEST == 7) {     // outer product with one scalar FFMA per two FFMA2 (the start-up's share)
#pragma unroll
            for (int j = 0; j < 14; ++j) {
                const u64 w = pk2(x[j], x[j]);
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    acc[4 * j + c] = fma2(w, q2[c], acc[4 * j + c]);
                    if (c & 1) x[15 - (j & 1)] = fmaf(x[15 - (j & 1)], a, b);
                }
            }
        } else if constexpr (TEST == 8) {     // outer product with one MUFU per 8 FFMA2
#pragma unroll
            for (int j = 0; j < 14; ++j) {
                const u64 w = pk2(x[j], x[j]);
#pragma unroll
                for (int c = 0; c < 4; ++c) acc[4 * j + c] = fma2(w, q2[c], acc[4 * j + c]);
                if (j & 1) x[15] = rsqrt_mufu(x[15]);
            }
        }
    }
    const long long t1 = clock64();
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) { float lo, hi; upk2(p[i], lo, hi); s += x[i] + lo + hi; }
#pragma unroll
    for (int i = 0; i < 56; ++i) { float lo, hi; upk2(acc[i], lo, hi); s += lo + hi; }
    if (s == 123.456f || iv == 0xdeadbeefu) sink[0] = s;              // keeps the arithmetic alive
    if ((tid & 31) == 0) {      // clock64 is the SM's cycle counter: (start, end, SM) per warp, combined per SM on the host
        unsigned sm;
        asm volatile("mov.u32 %0, %%smid;" : "=r"(sm));
        long long *c = cycles + 3 * (blockIdx.x * (blockDim.x / 32) + (tid >> 5));
        c[0] = t0; c[1] = t1; c[2] = (long long)sm;
    }
}

// FP32-pipe (MUFU for test 5) lane-operations per warp-lane and trip, and warp instructions per trip, of each test
const struct { double lane_ops; int instr; const char *name; } kTests[] = {
    {64, 64, "scalar FFMA"}, {128, 64, "FFMA2 (scalar-broadcast multiplier)"}, {128, 64, "FADD2"},
    {112, 56, "outer product FFMA2 (product form hot loop)"}, {224, 112, "FADD2 + FFMA2 chain step (chain form hot loop)"},
    {32, 64, "MUFU.SIN (sin.approx: FMUL.RZ + MUFU)"}, {112, 112, "outer product FFMA2 + 1 LOP3 each"},
    {140, 84, "outer product FFMA2 + 1 scalar FFMA per 2"}, {112, 63, "outer product FFMA2 + 1 MUFU.RSQ per 8"},
};
constexpr int kNumTests = sizeof(kTests) / sizeof(kTests[0]);

// MUFU.SIN error on (0, 1/2] turns against double: n points t_i = (i + 1/2) / (2 n); max |e|, sum e, sum e^2 per block
__global__ void mufu_err_kernel(int n, double *__restrict__ out)
{
    double mx = 0.0, s1 = 0.0, s2 = 0.0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const float t = (float)(((double)i + 0.5) / (2.0 * n));
        const double e = (double)sin_mufu(t * 6.28318530717958648f) - sin(6.283185307179586476925 * (double)t);
        mx = fmax(mx, fabs(e)); s1 += e; s2 += e * e;
    }
    __shared__ double sm[3][256];
    sm[0][threadIdx.x] = mx; sm[1][threadIdx.x] = s1; sm[2][threadIdx.x] = s2;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int i = 1; i < (int)blockDim.x; ++i) { sm[0][0] = fmax(sm[0][0], sm[0][i]); sm[1][0] += sm[1][i]; sm[2][0] += sm[2][i]; }
        out[3 * blockIdx.x] = sm[0][0]; out[3 * blockIdx.x + 1] = sm[1][0]; out[3 * blockIdx.x + 2] = sm[2][0];
    }
}

// MUFU.RSQ relative error on n points x_i = 4^((i + 1/2) / n) of [1, 4) (the exponent is handled exactly, so this is the
// whole error curve; log-uniform = how the mantissas of squared distances spread): e = rsqrt.approx(x) sqrt(x) - 1
__global__ void mufu_rsq_err_kernel(int n, double *__restrict__ out)
{
    double mx = 0.0, s1 = 0.0, s2 = 0.0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const float x = (float)exp2(2.0 * ((double)i + 0.5) / (double)n);
        const double e = (double)rsqrt_mufu(x) * sqrt((double)x) - 1.0;
        mx = fmax(mx, fabs(e)); s1 += e; s2 += e * e;
    }
    __shared__ double sm[3][256];
    sm[0][threadIdx.x] = mx; sm[1][threadIdx.x] = s1; sm[2][threadIdx.x] = s2;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int i = 1; i < (int)blockDim.x; ++i) { sm[0][0] = fmax(sm[0][0], sm[0][i]); sm[1][0] += sm[1][i]; sm[2][0] += sm[2][i]; }
        out[3 * blockIdx.x] = sm[0][0]; out[3 * blockIdx.x + 1] = sm[1][0]; out[3 * blockIdx.x + 2] = sm[2][0];
    }
}

template <int T>
cudaError_t launch(int blocks, int ctas_per_sm, int iters, const float *init, long long *cyc, float *sink, cudaStream_t st)
{
    int fit = 0;      // the rate is computed for ctas_per_sm concurrent CTAs: they must all be resident
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&fit, pipe_kernel<T>, 128, 0);
    if (e != cudaSuccess) return e;
    if (fit < ctas_per_sm) return cudaErrorLaunchOutOfResources;
    pipe_kernel<T><<<blocks, 128, 0, st>>>(iters, init, cyc, sink);
    return cudaGetLastError();
}
}  // namespace

extern "C" {

int debye_pipe_bench_count(void) { return kNumTests; }
const char *debye_pipe_bench_name(int test) { return (test >= 0 && test < kNumTests) ? kTests[test].name : nullptr; }

int debye_pipe_bench(int test, int ctas_per_sm, int iters, double *lane_ops_per_clk_per_sm, double *cycles_per_instr, debye_stream_t stream_)
{
    cudaStream_t st = (cudaStream_t)stream_;
    if (test < 0 || test >= kNumTests || ctas_per_sm < 1 || ctas_per_sm > 4 || iters < 1 || !lane_ops_per_clk_per_sm) return DEBYE_EINVAL;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return DEBYE_ECUDA;
    const int blocks = sms * ctas_per_sm, warps = blocks * 4;
    long long *cyc = nullptr; float *sink = nullptr, *init = nullptr;
    if (cudaMalloc(&cyc, sizeof(long long) * 3 * warps) != cudaSuccess) return DEBYE_ENOMEM;
    if (cudaMalloc(&sink, 4) != cudaSuccess) { cudaFree(cyc); return DEBYE_ENOMEM; }
    if (cudaMalloc(&init, 64 * 4) != cudaSuccess) { cudaFree(cyc); cudaFree(sink); return DEBYE_ENOMEM; }
    {
        float hinit[64];
        hinit[0] = 1.0000001f; hinit[1] = 1e-9f;
        for (int i = 2; i < 64; ++i) hinit[i] = 1e-9f * (float)(3 * i + 1);
        cudaMemcpyAsync(init, hinit, sizeof(hinit), cudaMemcpyHostToDevice, st);
        cudaStreamSynchronize(st);
    }
    cudaError_t e = cudaSuccess;
    for (int rep = 0; rep < 2 && e == cudaSuccess; ++rep) {      // the first launch warms the instruction cache
        switch (test) {
            case 0: e = launch<0>(blocks, ctas_per_sm, iters, init, cyc, sink, st); break;
            case 1: e = launch<1>(blocks, ctas_per_sm, iters, init, cyc, sink, st); break;
            case 2: e = launch<2>(blocks, ctas_per_sm, iters, init, cyc, sink, st); break;
            case 3: e = launch<3>(blocks, ctas_per_sm, iters, init, cyc, sink, st); break;
            case 4: e = launch<4>(blocks, ctas_per_sm, iters, init, cyc, sink, st); break;
            case 5: e = launch<5>(blocks, ctas_per_sm, iters, init, cyc, sink, st); break;
            case 6: e = launch<6>(blocks, ctas_per_sm, iters, init, cyc, sink, st); break;
            case 7: e = launch<7>(blocks, ctas_per_sm, iters, init, cyc, sink, st); break;
            default: e = launch<8>(blocks, ctas_per_sm, iters, init, cyc, sink, st); break;
        }
    }
    long long *h = new long long[3 * warps];
    if (e == cudaSuccess) e = cudaMemcpyAsync(h, cyc, sizeof(long long) * 3 * warps, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(cyc); cudaFree(sink); cudaFree(init);
    if (e != cudaSuccess) { delete[] h; (void)cudaGetLastError(); return e == cudaErrorLaunchOutOfResources ? DEBYE_EUNSUPPORTED : DEBYE_ECUDA; }
    // per SM: lane-operations of the warps that ran there / (last end - first start); the block scheduler need not place
    // exactly ctas_per_sm CTAs on every SM, so only SMs that held exactly ctas_per_sm x 4 warps are averaged
    constexpr int MAXSM = 1024;
    long long lo[MAXSM], hi[MAXSM]; int cnt[MAXSM];
    for (int i = 0; i < MAXSM; ++i) { lo[i] = 0x7fffffffffffffffLL; hi[i] = 0; cnt[i] = 0; }
    for (int i = 0; i < warps; ++i) {
        const int sm = (int)h[3 * i + 2];
        if (sm < 0 || sm >= MAXSM) continue;
        if (h[3 * i] < lo[sm]) lo[sm] = h[3 * i];
        if (h[3 * i + 1] > hi[sm]) hi[sm] = h[3 * i + 1];
        ++cnt[sm];
    }
    delete[] h;
    double rate = 0.0, cpi = 0.0; int used = 0;
    for (int i = 0; i < MAXSM; ++i) {
        if (cnt[i] != 4 * ctas_per_sm) continue;
        const double cyc_sm = (double)(hi[i] - lo[i]);
        rate += kTests[test].lane_ops * 32.0 * cnt[i] * (double)iters / cyc_sm;
        cpi += cyc_sm / ((double)iters * kTests[test].instr * (double)ctas_per_sm);     // one scheduler serves ctas_per_sm warps
        ++used;
    }
    if (used == 0) return DEBYE_EUNSUPPORTED;
    *lane_ops_per_clk_per_sm = rate / used;
    if (cycles_per_instr) *cycles_per_instr = cpi / used;
    return DEBYE_OK;
}

static int mufu_error(int which, int n, double *max_abs, double *rms, double *mean, debye_stream_t stream_)
{
    cudaStream_t st = (cudaStream_t)stream_;
    if (n < 1 || !max_abs || !rms || !mean) return DEBYE_EINVAL;
    const int blocks = 64;
    double *d = nullptr, h[3 * 64];
    if (cudaMalloc(&d, sizeof(h)) != cudaSuccess) return DEBYE_ENOMEM;
    if (which == 0) mufu_err_kernel<<<blocks, 256, 0, st>>>(n, d);
    else mufu_rsq_err_kernel<<<blocks, 256, 0, st>>>(n, d);
    cudaError_t e = cudaMemcpyAsync(h, d, sizeof(h), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(d);
    if (e != cudaSuccess) return DEBYE_ECUDA;
    double mx = 0, s1 = 0, s2 = 0;
    for (int i = 0; i < blocks; ++i) { if (h[3 * i] > mx) mx = h[3 * i]; s1 += h[3 * i + 1]; s2 += h[3 * i + 2]; }
    *max_abs = mx; *mean = s1 / n; *rms = sqrt(s2 / n);
    return DEBYE_OK;
}
int debye_mufu_sin_error(int n, double *max_abs, double *rms, double *mean, debye_stream_t stream) { return mufu_error(0, n, max_abs, rms, mean, stream); }
int debye_mufu_rsq_error(int n, double *max_rel, double *rms, double *mean, debye_stream_t stream) { return mufu_error(1, n, max_rel, rms, mean, stream); }

}  // extern "C"
