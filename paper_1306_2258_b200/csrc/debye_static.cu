// debye_static.cu -- debye_profile_static: the profile of ONE small structure with NO allocation (include/debye.h).
//
// Every other entry point takes its scratch (per-CTA FP64 records, plan, sorted copy) from a workspace that the library
// cudaMallocs and grows on demand, or that the caller sets.  Callers that may not allocate -- code under CUDA graph capture, a
// tight serving loop, a harness that forbids cudaMalloc -- get this entry point instead: it launches the one-launch kernel of
// debye_small.cuh (sort, product-form pairs, grid barrier, FP64 reduction, telescoping and form-factor epilogue in a single
// cooperative launch) with its records in the file-scope array below, a fixed part of the library's
// device image.  No cudaMalloc, cudaFree, event or stream creation, here or in anything it calls; inputs and the output are
// the caller's.
//
// The array: DEBYE_STATIC_SCRATCH_BYTES = (256 + 36) records x 128 slots x 8 bytes = 299 008 bytes, held by every GPU that
// loads this translation unit's module until the process exits.  It bounds the problem: N <= 2048 atoms, T <= 8 types, at most
// 128 non-zero q values on a grid q_k = (k + koff) dq (koff 0 or 1, promised by the caller's DEBYE_QHINT flags: q is device
// memory the host may not read), and a grid of at most 256 CTAs (one per SM; 148 on B200).
//
// In HOST code the name of a __device__ array is a host-side stand-in, not a device address: a kernel handed
// `debye_static_scratch` itself would fault (or, where the GPU can reach host memory, scribble somewhere else).  Its device
// address is looked up once per device, with that device current, by cudaGetSymbolAddress (static_setup) and it is that
// pointer the kernel gets.
//
// Contents: every record the kernel's final stage reads was written earlier in the SAME launch (a CTA writes one record per
// type pair of its unit range; the final stage reads exactly the CTAs that own units of the type pair, debye_small.cuh
// step 4), so nothing has to start at zero and nothing is cleared; the array keeps the last call's records.  All calls on one
// GPU share it: calls on one stream are ordered by the stream; calls that can overlap on the GPU (different streams without
// an event between them, two host threads on two streams) RACE on the records and give wrong profiles -- order them.
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>
#include <mutex>
#include "../../include/debye.h"
#include "debye_registry.h"
#include "debye_small.cuh"

static_assert(DEBYE_STATIC_MAX_ATOMS == DEBYE_SMALL_NMAX && DEBYE_STATIC_MAX_TYPES == DEBYE_SMALL_TMAX, "limits of debye_small_kernel");
static_assert(DEBYE_STATIC_SCRATCH_BYTES == (size_t)(DEBYE_STATIC_MAX_GRID + DEBYE_SMALL_TP) * DEBYE_KMAX_F32 * 8, "records of the largest case");

// the scratch of every debye_profile_static call on this GPU: per-CTA FP64 records, records[(cta + type pair)][K]
static __device__ __align__(256) unsigned char debye_static_scratch[DEBYE_STATIC_SCRATCH_BYTES];

namespace {

constexpr int MAX_DEV = 64;
struct StaticDev {
    double *scratch = nullptr;      // DEVICE address of debye_static_scratch on this GPU (cudaGetSymbolAddress), never the host symbol
    int sms = 0;
    bool attr_set[DEBYE_KMAX_F32 / 8 + 1] = {};
};
StaticDev g_sdev[MAX_DEV];
std::mutex g_smu;
thread_local int g_static_cuda = 0;
thread_local char g_static_msg[256] = "";

int refuse(int code, const char *fmt, int a = 0, int b = 0)
{
    snprintf(g_static_msg, sizeof(g_static_msg), fmt, a, b);
    return code;
}
int cuda_fail(cudaError_t e, const char *what)
{
    g_static_cuda = (int)e;
    snprintf(g_static_msg, sizeof(g_static_msg), "debye_profile_static: %s failed: %s", what, cudaGetErrorString(e));
    (void)cudaGetLastError();
    return DEBYE_ECUDA;
}

// once per device, with that device current: SM count and the device address of the scratch array
int static_setup(StaticDev **out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
    if (dev < 0 || dev >= MAX_DEV) return refuse(DEBYE_EUNSUPPORTED, "debye_profile_static: device ordinal %d beyond the %d this build tracks", dev, MAX_DEV);
    StaticDev *s = &g_sdev[dev];
    std::lock_guard<std::mutex> lock(g_smu);
    if (!s->scratch) {
        int sms = 0;
        if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return cuda_fail(e, "cudaDeviceGetAttribute");
        int coop = 0;
        if ((e = cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev)) != cudaSuccess) return cuda_fail(e, "cudaDeviceGetAttribute");
        if (!coop) return refuse(DEBYE_EUNSUPPORTED, "debye_profile_static: device %d has no cooperative launch", dev);
        void *p = nullptr;
        if ((e = cudaGetSymbolAddress(&p, debye_static_scratch)) != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(debye_static_scratch)");
        if (!p || ((uintptr_t)p & 255)) return refuse(DEBYE_ECUDA, "debye_profile_static: scratch symbol address missing or misaligned");
        s->sms = sms;
        s->scratch = (double *)p;
    }
    *out = s;
    return DEBYE_OK;
}

// grid class promised by the hint flags: 0 for q_k = k dq from q_0 = 0, 1 for q_k = (k + 1) dq, negative otherwise
int static_hint_class(uint32_t flags)
{
    if (!(flags & DEBYE_QHINT) || !(flags & DEBYE_QHINT_UNIFORM)) return -1;
    const uint32_t st = flags & (DEBYE_QHINT_START0 | DEBYE_QHINT_STARTDQ);
    if (st == DEBYE_QHINT_START0) return 0;
    if (st == DEBYE_QHINT_STARTDQ) return 1;
    return -1;
}

}  // namespace

extern "C" {

int debye_profile_static(const float *xyz, const int32_t *type, int32_t N, const float *fftab, int32_t T, const float *q, int32_t M, double *I_out, uint32_t flags,
                         debye_stream_t stream_)
{
    g_static_msg[0] = 0;
    if (!xyz || !type || !fftab || !q || !I_out) return refuse(DEBYE_EINVAL, "debye_profile_static: null pointer");
    if (N < 1 || T < 1 || M < 1) return refuse(DEBYE_EINVAL, "debye_profile_static: N, T, M must be at least 1");
    const uint32_t known = DEBYE_SINC_RECUR | DEBYE_QHINT | DEBYE_QHINT_UNIFORM | DEBYE_QHINT_START0 | DEBYE_QHINT_STARTDQ;
    if (flags & ~(known | DEBYE_FP64 | DEBYE_SINC_MUFU | DEBYE_SINC_ACCURATE)) return refuse(DEBYE_EINVAL, "debye_profile_static: unknown flag bits");
    if (flags & ~known)
        return refuse(DEBYE_EUNSUPPORTED, "debye_profile_static: only the recurrence kernel exists without allocation (flags: grid hint, optionally DEBYE_SINC_RECUR)");
    const int cls = static_hint_class(flags);
    if (cls < 0)
        return refuse(DEBYE_EUNSUPPORTED,
                      "debye_profile_static: needs DEBYE_QHINT | DEBYE_QHINT_UNIFORM | DEBYE_QHINT_START0 or _STARTDQ (debye_q_hint): the grid must be q_k = (k + koff) dq, koff 0 or 1");
    if (N > DEBYE_STATIC_MAX_ATOMS) return refuse(DEBYE_EUNSUPPORTED, "debye_profile_static: N = %d atoms beyond the maximum of %d of the static scratch", N, DEBYE_STATIC_MAX_ATOMS);
    if (T > DEBYE_STATIC_MAX_TYPES) return refuse(DEBYE_EUNSUPPORTED, "debye_profile_static: T = %d types beyond the maximum of %d of the static scratch", T, DEBYE_STATIC_MAX_TYPES);
    const int n_idx = M - (cls == 0 ? 1 : 0);                      // non-zero q values = chain indices
    if (n_idx < 1) return refuse(DEBYE_EUNSUPPORTED, "debye_profile_static: the grid has no non-zero q (M = %d starting at 0)", M);
    if (n_idx > DEBYE_STATIC_MAX_Q)
        return refuse(DEBYE_EUNSUPPORTED, "debye_profile_static: %d non-zero q values beyond the maximum of %d of the static scratch", n_idx, DEBYE_STATIC_MAX_Q);

    StaticDev *s = nullptr;
    int st = static_setup(&s);
    if (st) return st;
    const int K = (debye::recur_slots(n_idx, 1) + 7) / 8 * 8;      // accumulators per thread: the instantiation of debye_small_kernel
    debye_small_fn fn = debye_get_small_kernel(K);
    if (!fn) return refuse(DEBYE_EUNSUPPORTED, "debye_profile_static: no kernel instantiation with %d accumulators", K);
    cudaError_t e;
    {
        std::lock_guard<std::mutex> lock(g_smu);
        if (!s->attr_set[K / 8]) {
            if ((e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)debye::debye_small_dyn_smem(DEBYE_SMALL_NMAX, DEBYE_SMALL_TMAX, DEBYE_KMAX_F32))) != cudaSuccess)
                return cuda_fail(e, "cudaFuncSetAttribute");
            s->attr_set[K / 8] = true;
        }
    }
    // the grid of the allocating path (debye_api.cu small_grid): at least ~6 units (one j atom x 128 i atoms) per CTA, one CTA
    // per SM at most -- the same unit ranges, hence the same bits -- and never more CTAs than the array has records for
    int64_t g = ((int64_t)N * N / (2 * DEBYE_IB) + 1) / 6;
    if (g > (int64_t)s->sms) g = s->sms;
    if (g > DEBYE_STATIC_MAX_GRID) g = DEBYE_STATIC_MAX_GRID;
    if (g < 1) g = 1;
    const int G = (int)g;
    const size_t need = ((size_t)G + (size_t)(T * (T + 1) / 2)) * K * 8;
    if (need > DEBYE_STATIC_SCRATCH_BYTES) return refuse(DEBYE_EUNSUPPORTED, "debye_profile_static: %d records needed, the static scratch holds fewer", G + T * (T + 1) / 2);

    cudaStream_t stream = (cudaStream_t)stream_;
    double *records = s->scratch;                                  // the DEVICE address; not the symbol
    int n = N, t = T, m = M, hc = cls, mode = 0;
    int32_t *n_out = nullptr;
    void *args[] = {(void *)&xyz, (void *)&type, (void *)&n, (void *)&t, (void *)&fftab, (void *)&q, (void *)&m, (void *)&hc, (void *)&records, (void *)&I_out, (void *)&mode, (void *)&n_out};
    if ((e = cudaLaunchCooperativeKernel((const void *)fn, dim3(G), dim3(DEBYE_IB), args, debye::debye_small_dyn_smem(N, T, K), stream)) != cudaSuccess)
        return cuda_fail(e, "cudaLaunchCooperativeKernel");
    return DEBYE_OK;
}

const char *debye_profile_static_error(void) { return g_static_msg; }

void debye_profile_static_limits(int32_t *max_atoms, int32_t *max_types, int32_t *max_nonzero_q, size_t *scratch_bytes)
{
    if (max_atoms) *max_atoms = DEBYE_STATIC_MAX_ATOMS;
    if (max_types) *max_types = DEBYE_STATIC_MAX_TYPES;
    if (max_nonzero_q) *max_nonzero_q = DEBYE_STATIC_MAX_Q;
    if (scratch_bytes) *scratch_bytes = DEBYE_STATIC_SCRATCH_BYTES;
}

}  // extern "C"
