// debye_api.cu -- the C ABI of libdebye (include/debye.h): validation, workspace, launch sequence.
//
// Launch sequence of one call (all on the caller's stream, no host synchronisation, no device->host reads):
//   debye_setup_kernel  (1 CTA)    type histogram, stable sort permutation, q analysis, unit prefix   S0/S1
//   debye_pack_kernel               gather into type-sorted float4                                     S0
//   debye_pairs_kernel<K, variant>  persistent grid, one or (automatic mode) two launches of which     S1-S6
//                                   the one not selected on the device exits immediately
//   debye_reduce_kernel             fixed-order FP64 sum of the per-CTA records                        S7
//   debye_epilogue_kernel           telescoping of the product form, form-factor epilogue              S7
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <cstddef>
#include <cmath>
#include <mutex>
#include <algorithm>
#include <vector>
#include "../../include/debye.h"
#include "debye_aux.cuh"
#include "debye_pairs.cuh"
#include "debye_plan.cuh"
#include "debye_registry.h"
#include "debye_peratom.cuh"
#include "debye_small.cuh"
#include "debye_peratom_recur.cuh"
#include "debye_peratom_small.cuh"

namespace {

thread_local int g_last_cuda = 0;
#define CU(call)                                   \
    do {                                           \
        cudaError_t e__ = (call);                  \
        if (e__ != cudaSuccess) {                  \
            g_last_cuda = (int)e__;                \
            return DEBYE_ECUDA;                    \
        }                                          \
    } while (0)

// Scratch shared by calls on different streams (the per-device workspace and staging buffer; a plan's own workspace): acquire
// before the first use in a call, release behind the last.  Same stream as the previous user: stream order is enough.
struct ScratchOrder { cudaEvent_t done = nullptr; cudaStream_t stream = nullptr; bool used = false; };
cudaError_t scratch_acquire(ScratchOrder &o, cudaStream_t stream)
{
    if (o.used && o.stream != stream) return cudaStreamWaitEvent(stream, o.done, 0);
    return cudaSuccess;
}
cudaError_t scratch_release(ScratchOrder &o, cudaStream_t stream)
{
    if (!o.done) { cudaError_t e = cudaEventCreateWithFlags(&o.done, cudaEventDisableTiming); if (e != cudaSuccess) return e; }
    o.stream = stream; o.used = true;
    return cudaEventRecord(o.done, stream);
}

// debye_q_hint: 1 = a uniform grid with a general start (neither 0 nor dq) is hinted as pieces too: the centred product form
// (measured on B200, 10 000 atoms x 101 q: 11.6 T pair.q/s) instead of the chain form of the recurrence (4.65 T)
#ifndef DEBYE_CENT_FOR_GENERAL_START
#define DEBYE_CENT_FOR_GENERAL_START 1
#endif
#ifndef DEBYE_MUFU_KMAX
#define DEBYE_MUFU_KMAX 112      // largest q-chunk of the MUFU kernel (choose())
#endif
static_assert(DEBYE_SETUP_MAXQ == DEBYE_MAX_Q, "the setup kernel stages the whole q grid in shared memory");
#ifndef DEBYE_PAS_CTAS_PER_SM
#define DEBYE_PAS_CTAS_PER_SM 1  // fused per-atom kernel for small structures: CTAs per SM of its cooperative grid
#endif
#ifndef DEBYE_PAS_UNITS
#define DEBYE_PAS_UNITS 6
#endif
#ifndef DEBYE_UNITS_PER_CTA
// grid_for: at least this many units (one j atom x 128 i atoms) per pairs CTA.  Measured on B200 with the product form, cfg2
// (G pair.q/s by units per CTA): 75 14 334, 100 14 631, 150 15 040, 250 15 160, 400 15 152, 800 14 854 (a single wave)
#define DEBYE_UNITS_PER_CTA 250.0
#endif
#ifndef DEBYE_PAR_UNITS_PER_CTA
#define DEBYE_PAR_UNITS_PER_CTA 250  // per-atom recurrence: units per pairs CTA (cfg2: 150 6 189, 250 6 270, 400 5 857 G pair.q/s)
#endif
#ifndef DEBYE_PA_PDL
#define DEBYE_PA_PDL 1           // per-atom launch chains with programmatic dependent launch (0: ordinary launches, for measurement)
#endif
constexpr int MAX_DEV = 64;
constexpr int64_t DEBYE_PACK_IN_SETUP = 16384;   // N x B up to which debye_setup_kernel also packs the coordinates
struct DevState {
    void *ws = nullptr; size_t ws_bytes = 0;          // library-owned scratch
    void *user_ws = nullptr; size_t user_bytes = 0;   // caller-owned scratch (debye_set_workspace)
    void *stage = nullptr; size_t stage_bytes = 0;    // device staging for the *_host entry points
    void *hstage = nullptr; size_t hstage_bytes = 0;  // pinned host staging: small inputs of the *_host entries travel as ONE copy
    int sms = 0;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;         // optional: recorded around the pairs launches
    // cross-stream ordering of the shared scratch (workspace, staging buffer): every call records ws_done behind its last
    // use; a call on another stream first makes its stream wait for it, so calls on different streams serialise on the
    // device instead of overwriting each other's records
    ScratchOrder order;
    int occ[6][33];                                   // cached CTAs/SM per (variant, K/4); 0 = unknown
    int occ_small[17][DEBYE_SMALL_TMAX + 1];          // the same for debye_small_kernel<8 i> with T types (N = 2048); 0 = unknown
};
DevState g_dev[MAX_DEV];
std::mutex g_mu;
std::mutex g_hstage_mu;                               // one *_host call at a time fills and drains the pinned staging buffer
bool g_atexit = false;
constexpr size_t HOST_ONE_COPY_MAX = 256 * 1024;      // inputs up to this size are gathered on the host and copied once

size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }



// launch with programmatic stream serialisation (PDL, debye_plan.cuh): the kernel must start with pdl_wait()
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, cudaStream_t stream, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = 0; cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

struct Choice { int variant; int K; int n_chunks; int alt_gate; };   // alt_gate: -1 always runs, 0 / 1 see debye_pairs_kernel

// q-chunking of each variant: how many accumulators a thread keeps (K) and how many passes over the pairs.
Choice choose(int variant, int M)
{
    Choice c; c.variant = variant; c.alt_gate = -1;
    if (variant == V_RECUR) {
        // M chain indices (worst case: grid starting at dq, or general start); residue-class chunks: a power of two
        int nc = 1;
        while (debye::recur_slots(M, nc) > DEBYE_KMAX_F32) nc *= 2;
        c.n_chunks = nc; c.K = debye::recur_slots(M, nc);
    } else {
        // MUFU: the pipelined loop needs K + ~75 registers and spills inside the loop above K = 112 (measured: M = 128 as one
        // chunk of 128 runs at 2.28 T pair.q/s on cfg5; two chunks repeat only the distance)
        int kmax = (variant == V_F64) ? DEBYE_KMAX_F64 : (variant == V_MUFU ? DEBYE_MUFU_KMAX : DEBYE_KMAX_F32);
        int nc = (M + kmax - 1) / kmax;
        int per = (M + nc - 1) / nc;
        c.n_chunks = nc; c.K = (per + 7) / 8 * 8;
    }
    return c;
}
// Recurrence launches: a grid that starts at q = 0 needs one chain index fewer (q = 0 is answered by the epilogue), which
// can save four accumulators or a whole chunk -- but only the device knows q.  When it pays, a second instantiation
// sized for M - 1 indices is launched as well and the device runs exactly one of the two (plan->recur_alt).
int recur_choices(Choice *out, int M)
{
    const Choice main_c = choose(V_RECUR, M);
    if (M >= 2) {
        Choice alt = choose(V_RECUR, M - 1);
        if (alt.n_chunks <= 2 && (alt.K < main_c.K || alt.n_chunks < main_c.n_chunks)) {
            alt.alt_gate = 1;
            out[0] = alt; out[1] = main_c; out[1].alt_gate = 0;
            return 2;
        }
    }
    out[0] = main_c;
    return 1;
}

struct Layout { size_t plan, perm, sorted, records, sums, total; };
Layout layout(int N, int B, int T, int M, int G_max, const Choice *ch, int nch)
{
    Layout L; size_t o = 0;
    L.plan = o; o += align_up(sizeof(DevPlan));
    L.perm = o; o += align_up((size_t)N * 4);
    L.sorted = o; o += align_up((size_t)N * B * 16);
    size_t rec = 0, sm = 0;
    for (int i = 0; i < nch; ++i) {
        size_t r = ((size_t)G_max + (size_t)B * (T * (T + 1) / 2) * ch[i].n_chunks) * ch[i].K * 8;
        size_t m = (size_t)B * (T * (T + 1) / 2) * ch[i].n_chunks * ch[i].K * 8;
        if (r > rec) rec = r;
        if (m > sm) sm = m;
    }
    L.records = o; o += align_up(rec);
    L.sums = o; o += align_up(sm);
    L.total = o;
    return L;
}

constexpr int MAX_CHOICES = 4;
// grid class promised by the caller's hint flags (debye_grid_class), -3 without a hint, -4 for a piecewise-uniform grid
int hint_class_of(uint32_t flags)
{
    if (!(flags & DEBYE_QHINT)) return -3;
    if (flags & DEBYE_QHINT_PIECES) return -4;
    if (!(flags & DEBYE_QHINT_UNIFORM)) return -2;
    if (flags & DEBYE_QHINT_START0) return 0;
    if (flags & DEBYE_QHINT_STARTDQ) return 1;
    return -1;
}
// piecewise-uniform hint: number of pieces and accumulators per thread, as (n << 8) | K / 8 (the setup kernel's argument)
int hint_pieces_of(uint32_t flags)
{
    if (!(flags & DEBYE_QHINT_PIECES)) return 0;
    return (int)((((flags >> DEBYE_QHINT_NPIECES_SHIFT) & 31u) + 1u) << 8) | (int)(((flags >> DEBYE_QHINT_PIECEK_SHIFT) & 31u) + 1u);
}
Choice cent_choice(uint32_t flags)
{
    const int hp = hint_pieces_of(flags);
    Choice c; c.variant = V_CENT; c.K = 8 * (hp & 255); c.n_chunks = hp >> 8; c.alt_gate = -1;
    return c;
}
// the one recurrence launch for a known grid class
int recur_choice_hinted(Choice *out, int M, int cls)
{
    Choice c[2];
    const int n = recur_choices(c, M);
    out[0] = (n == 2 && cls == 0) ? c[0] : c[n - 1];      // the launch sized for M - 1 indices only when q[0] == 0
    out[0].alt_gate = -1;
    return 1;
}
// centred form for ONE uniform run of M points (a uniform grid with a general start): its pieces follow from M alone
// (debye_find_pieces: equal pieces of at most DEBYE_PIECE_KCAP points); false if that needs more than DEBYE_MAX_PIECES
bool cent_choice_uniform(Choice *out, int M)
{
    const int np = (M + DEBYE_PIECE_KCAP - 1) / DEBYE_PIECE_KCAP, per = (M + np - 1) / np;
    if (np > DEBYE_MAX_PIECES) return false;
    out->variant = V_CENT; out->K = (per + 7) / 8 * 8; out->n_chunks = np; out->alt_gate = -1;
    if (out->K < 8) out->K = 8;
    return true;
}
int variants_for(uint32_t flags, Choice *out, int M, int *is_auto)
{
    *is_auto = 0;
    const int cls = hint_class_of(flags);
    if (flags & DEBYE_FP64) { out[0] = choose(V_F64, M); return 1; }
    if (flags & DEBYE_SINC_MUFU) { out[0] = choose(V_MUFU, M); return 1; }
    if (flags & DEBYE_SINC_RECUR) return (cls >= -1) ? recur_choice_hinted(out, M, cls) : recur_choices(out, M);
    if (flags & DEBYE_SINC_ACCURATE) { out[0] = choose(V_ACCURATE, M); return 1; }
    if (flags & DEBYE_SINC_CENTRED) { out[0] = cent_choice(flags); return 1; }      // validate(): only with a pieces hint
    *is_auto = 1;
    if (cls == -4) { out[0] = cent_choice(flags); return 1; }         // hinted: piecewise uniform, the centred product form
    if (cls == -2) { out[0] = choose(V_MUFU, M); return 1; }          // hinted: not uniform
    if (cls >= -1) return recur_choice_hinted(out, M, cls);           // hinted: uniform
    // no hint: every instantiation the grid could need is launched and the device runs one of them -- the recurrence (grids
    // from 0 or dq: product form), the centred form (uniform with a general start), the MUFU kernel (anything else)
    int n = recur_choices(out, M);
    if (cent_choice_uniform(&out[n], M)) ++n;
    out[n++] = choose(V_MUFU, M);
    return n;
}

int validate(const void *xyz, const void *type, int N, int B, const void *tab, int T, const void *q, int M, const void *out, uint32_t flags)
{
    if (!xyz || !type || !q || !out) return DEBYE_EINVAL;
    if (!tab) return DEBYE_EINVAL;
    if (N < 1 || M < 1 || T < 1 || B < 1 || T > DEBYE_MAX_TYPES || M > DEBYE_MAX_Q) return DEBYE_EINVAL;
    const uint32_t piece_fields = (31u << DEBYE_QHINT_NPIECES_SHIFT) | (31u << DEBYE_QHINT_PIECEK_SHIFT);
    uint32_t known = DEBYE_FP64 | DEBYE_SINC_MUFU | DEBYE_SINC_RECUR | DEBYE_SINC_ACCURATE | DEBYE_SINC_CENTRED | DEBYE_QHINT | DEBYE_QHINT_UNIFORM |
                     DEBYE_QHINT_START0 | DEBYE_QHINT_STARTDQ | DEBYE_QHINT_PIECES | piece_fields;
    if (flags & ~known) return DEBYE_EINVAL;
    uint32_t s = flags & (DEBYE_SINC_MUFU | DEBYE_SINC_RECUR | DEBYE_SINC_ACCURATE | DEBYE_SINC_CENTRED);
    if (s & (s - 1)) return DEBYE_EINVAL;
    if ((flags & DEBYE_FP64) && s) return DEBYE_EINVAL;
    {   // grid hint: sub-bits only with DEBYE_QHINT, start bits only for uniform grids and not both
        const uint32_t sub = flags & (DEBYE_QHINT_UNIFORM | DEBYE_QHINT_START0 | DEBYE_QHINT_STARTDQ), st2 = flags & (DEBYE_QHINT_START0 | DEBYE_QHINT_STARTDQ);
        if (sub && !(flags & DEBYE_QHINT)) return DEBYE_EINVAL;
        if (st2 && !(flags & DEBYE_QHINT_UNIFORM)) return DEBYE_EINVAL;
        if (st2 == (DEBYE_QHINT_START0 | DEBYE_QHINT_STARTDQ)) return DEBYE_EINVAL;
        // piecewise-uniform hint: excludes the uniform bits; its fields (pieces - 1, K / 8 - 1) only with it, at most 32 pieces and K <= 128
        if ((flags & DEBYE_QHINT_PIECES) && (!(flags & DEBYE_QHINT) || sub)) return DEBYE_EINVAL;
        if (!(flags & DEBYE_QHINT_PIECES) && (flags & piece_fields)) return DEBYE_EINVAL;
        if ((flags & DEBYE_QHINT_PIECES) && ((((flags >> DEBYE_QHINT_NPIECES_SHIFT) & 31u) >= DEBYE_MAX_PIECES) || (((flags >> DEBYE_QHINT_PIECEK_SHIFT) & 31u) >= 16u)))
            return DEBYE_EINVAL;
        // the centred product form needs the pieces: the host sizes the launch from them
        if ((flags & DEBYE_SINC_CENTRED) && !(flags & DEBYE_QHINT_PIECES)) return DEBYE_EUNSUPPORTED;
    }
    if (N > (1 << 24)) return DEBYE_EUNSUPPORTED;
    if ((int64_t)N * B > ((int64_t)1 << 31)) return DEBYE_EUNSUPPORTED;
    return DEBYE_OK;
}

int dev_state(DevState **st)
{
    int dev = 0;
    CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEV) return DEBYE_EUNSUPPORTED;
    DevState *s = &g_dev[dev];
    if (s->sms == 0) {
        int sms = 0;
        CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        s->sms = sms;
        memset(s->occ, 0, sizeof(s->occ));
        memset(s->occ_small, 0, sizeof(s->occ_small));
    }
    *st = s;
    return DEBYE_OK;
}

// Grid of the pairs kernel: resident CTAs (SMs x occupancy) times a number of waves.  The warp schedulers favour one of
// the CTAs that share an SM, so with exactly one wave the favoured CTA finishes ~30 % early and its partner runs the tail
// alone (measured); more waves let the hardware block scheduler refill the SM.  Each extra CTA costs
// one prologue, one FP64 flush and one more record for the final kernel, so the count is bounded by the work available
// (estimated from N alone: the host never sees the type histogram): at least DEBYE_UNITS_PER_CTA units (one j atom x 128 i
// atoms) per CTA, at most 16 waves -- cfg2 with the product form: 3 waves of 3 CTAs per SM; flat beyond 4 waves on the large configs.
int grid_for(DevState *s, const Choice &c, int N, int B, int *G, bool weighted = false)
{
    int &o = s->occ[c.variant][c.K / 4];
    if (o == 0) {
        debye_pairs_fn fn = debye_get_pairs_kernel(c.variant, c.K, false);      // the weighted twin has the same launch bounds
        if (!fn) return DEBYE_EUNSUPPORTED;
        int nb = 0;
        CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, fn, DEBYE_IB, 0));
        if (nb < 1) nb = 1;
        o = nb;
    }
    const int resident = s->sms * o;
    const double units = (double)B * c.n_chunks * ((double)N * (double)N / (2.0 * DEBYE_IB));   // j atoms x rows, all type pairs
    // the direct variants (one MUFU.SIN / sinf / double sin per term) keep 150: their units take 5 to 50 times longer, and the MUFU
    // kernel measured 3 237 G pair.q/s on cfg2 with 150 units per CTA against 3 120 G with 250
    const double units_per_cta = (c.variant == V_RECUR || c.variant == V_CENT) ? DEBYE_UNITS_PER_CTA : 150.0;
    int waves = (int)(units / ((double)resident * units_per_cta));
    if (waves < 1) waves = 1;
    if (waves > 16) waves = 16;
    *G = resident * waves;
    return DEBYE_OK;
}

void shutdown_all()
{
    for (int d = 0; d < MAX_DEV; ++d) {
        if (g_dev[d].ws || g_dev[d].stage || g_dev[d].hstage) {
            int cur = 0;
            if (cudaGetDevice(&cur) != cudaSuccess) return;
            if (cudaSetDevice(d) != cudaSuccess) continue;
            if (g_dev[d].ws) cudaFree(g_dev[d].ws);
            if (g_dev[d].stage) cudaFree(g_dev[d].stage);
            if (g_dev[d].hstage) cudaFreeHost(g_dev[d].hstage);
            g_dev[d].ws = g_dev[d].stage = g_dev[d].hstage = nullptr; g_dev[d].ws_bytes = g_dev[d].stage_bytes = g_dev[d].hstage_bytes = 0;
            cudaSetDevice(cur);
        }
    }
}

int ensure(void **ptr, size_t *have, size_t need)
{
    if (*have >= need) return DEBYE_OK;
    if (*ptr) { CU(cudaFree(*ptr)); *ptr = nullptr; *have = 0; }
    size_t want = need + need / 4;
    cudaError_t e = cudaMalloc(ptr, want);
    if (e != cudaSuccess) { (void)cudaGetLastError(); g_last_cuda = (int)e; *ptr = nullptr; return DEBYE_ENOMEM; }
    *have = want;
    if (!g_atexit) { g_atexit = true; atexit(shutdown_all); }
    return DEBYE_OK;
}

}  // namespace (reopened below)
// A plan owns the device-resident result of the setup step (DevPlan, sort permutation) and copies of q and the weights, so
// that repeated profiles of one molecule (only the coordinates change: refinement loops) skip the sort
// and launch exactly the one pairs instantiation the grid needs.
struct debye_plan {
    int N, B, T, M, device;
    uint32_t flags;              // the caller's flags with the grid hint resolved at creation
    char *buf;                   // one allocation: DevPlan | perm[N] | q[M] | weight[N] | type[N] | workspace
    DevPlan *plan; int32_t *perm; float *q; float *weight; int32_t *type;
    char *ws; size_t ws_bytes;   // the plan's own scratch: plans on different streams run concurrently
    ScratchOrder order;          // ... and one plan used on several streams serialises on the device
};
namespace {

// One launch for one small structure (debye_small.cuh): single structure, unweighted, not sharded, N <= 2048, T <= 8, and a
// grid hint that promises q_k = (k + koff) dq with at most 128 chain indices (the kernel verifies the hint; NaN otherwise).
bool small_eligible(int N, int B, int T, int M, uint32_t flags, const float *weight, int shard_world)
{
    if (B != 1 || weight || shard_world != 1 || N > DEBYE_SMALL_NMAX || T > DEBYE_SMALL_TMAX) return false;
    if (flags & (DEBYE_FP64 | DEBYE_SINC_MUFU | DEBYE_SINC_ACCURATE)) return false;
    const int cls = hint_class_of(flags);
    if (cls != 0 && cls != 1) return false;
    const int n_idx = M - (cls == 0 ? 1 : 0);
    return n_idx >= 1 && n_idx <= DEBYE_KMAX_F32;
}
int small_K(int M, uint32_t flags) { return (debye::recur_slots(M - (hint_class_of(flags) == 0 ? 1 : 0), 1) + 7) / 8 * 8; }
int small_grid(DevState *ds, int N, int T, int K, int *G)
{
    int &o = ds->occ_small[K / 8][T];
    debye_small_fn fn = debye_get_small_kernel(K);
    if (!fn) return DEBYE_EUNSUPPORTED;
    if (o == 0) {
        // dynamic shared memory up to the largest case (T = 8, K = 128 sums / 2048 atoms); opt in once
        CU(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)debye::debye_small_dyn_smem(DEBYE_SMALL_NMAX, DEBYE_SMALL_TMAX, DEBYE_KMAX_F32)));
        int nb = 0;
        CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, fn, DEBYE_IB, debye::debye_small_dyn_smem(DEBYE_SMALL_NMAX, T, K)));
        o = nb < 1 ? 1 : nb;
    }
    // one wave at most; at least ~6 units (j atoms x 128 i atoms) per CTA, estimated from N alone
    const int64_t units = (int64_t)N * N / (2 * DEBYE_IB) + 1;
    // one CTA per SM at most (measured on B200, 1000 and 2000 atoms: 28.8 / 37.0 us per profile with 148 CTAs, 29.2 / 37.4
    // with 296, 33.3 / 42.9 with 592: every CTA pays the sort, and the final stage grows with the number of records)
    int64_t g = units / 6;
    if (g > (int64_t)ds->sms) g = (int64_t)ds->sms;
    if (g > DEBYE_SMALL_GMAX) g = DEBYE_SMALL_GMAX;            // what the kernel's shared-memory layout of the final stage holds
    if (g < 1) g = 1;
    *G = (int)g;
    return DEBYE_OK;
}
size_t small_ws_bytes(int T, int K, int G) { return align_up(((size_t)G + (size_t)(T * (T + 1) / 2)) * K * 8); }

int run_small(DevState *ds, const float *xyz, const int32_t *type, int N, const float *fftab, int T, const float *q, int M, double *out, int32_t *n_out,
              uint32_t flags, cudaStream_t stream, int mode, debye_plan *pre, std::unique_lock<std::mutex> &lock)
{
    const int K = small_K(M, flags);
    int G = 0, st;
    if ((st = small_grid(ds, N, T, K, &G))) return st;
    const size_t need = small_ws_bytes(T, K, G);
    char *ws;
    ScratchOrder *order = &ds->order;
    if (pre && pre->ws) { if (pre->ws_bytes < need) return DEBYE_ENOMEM; ws = pre->ws; order = &pre->order; }
    else if (ds->user_ws) { if (ds->user_bytes < need) return DEBYE_ENOMEM; ws = (char *)ds->user_ws; }
    else { if ((st = ensure(&ds->ws, &ds->ws_bytes, need))) return st; ws = (char *)ds->ws; }
    cudaEvent_t ev0 = ds->ev0, ev1 = ds->ev1;
    if (pre && pre->ws) lock.unlock();             // nothing shared with other calls from here on
    CU(scratch_acquire(*order, stream));
    debye_small_fn fn = debye_get_small_kernel(K);
    if (ev0) CU(cudaEventRecord(ev0, stream));
    {   // cooperative launch: the kernel has a grid-wide barrier (G is at most one resident wave, small_grid)
        int hc = hint_class_of(flags);
        double *rec = (double *)ws;
        void *args[] = {(void *)&xyz, (void *)&type, (void *)&N, (void *)&T, (void *)&fftab, (void *)&q, (void *)&M, (void *)&hc, (void *)&rec, (void *)&out, (void *)&mode, (void *)&n_out};
        CU(cudaLaunchCooperativeKernel((const void *)fn, dim3(G), dim3(DEBYE_IB), args, debye::debye_small_dyn_smem(N, T, K), stream));
    }
    if (ev1) CU(cudaEventRecord(ev1, stream));
    CU(scratch_release(*order, stream));
    CU(cudaGetLastError());
    return DEBYE_OK;
}

// mode 0: I_out[B][M]; mode 1: S_out[B][n_tp][M] (+ n_out)
int run(const float *xyz, const int32_t *type, int N, int B, const float *fftab, int T, const float *q, int M, double *out, int32_t *n_out,
        uint32_t flags, cudaStream_t stream, int mode, const float *weight = nullptr, debye_plan *pre = nullptr, int shard_rank = 0,
        int shard_world = 1)
{
    int st = validate(xyz, type, N, B, mode == 0 ? (const void *)fftab : (const void *)q, T, q, M, out, flags);
    if (st) return st;
    std::unique_lock<std::mutex> lock(g_mu);
    DevState *ds;
    if ((st = dev_state(&ds))) return st;
    if (small_eligible(N, B, T, M, flags, weight, shard_world) && (!pre || pre->type))
        return run_small(ds, xyz, pre ? pre->type : type, N, fftab, T, q, M, out, n_out, flags, stream, mode, pre, lock);
    Choice ch[MAX_CHOICES]; int is_auto = 0;
    const int nch = variants_for(flags, ch, M, &is_auto);
    int G[MAX_CHOICES] = {0, 0, 0, 0}, Gmax = 0;
    for (int i = 0; i < nch; ++i) { if ((st = grid_for(ds, ch[i], N, B, &G[i]))) return st; if (G[i] > Gmax) Gmax = G[i]; }
    const Layout L = layout(N, B, T, M, Gmax, ch, nch);
    char *ws;
    ScratchOrder *order = &ds->order;
    if (pre && pre->ws) { if (pre->ws_bytes < L.total) return DEBYE_ENOMEM; ws = pre->ws; order = &pre->order; }
    else if (ds->user_ws) { if (ds->user_bytes < L.total) return DEBYE_ENOMEM; ws = (char *)ds->user_ws; }
    else { if ((st = ensure(&ds->ws, &ds->ws_bytes, L.total))) return st; ws = (char *)ds->ws; }
    const cudaEvent_t ev0 = ds->ev0, ev1 = ds->ev1;
    const int sms = ds->sms;
    if (pre && pre->ws) lock.unlock();             // a plan's own scratch: nothing shared with other calls from here on
    CU(scratch_acquire(*order, stream));
    DevPlan *plan = pre ? pre->plan : (DevPlan *)(ws + L.plan);
    int32_t *perm = pre ? pre->perm : (int32_t *)(ws + L.perm);
    float4 *sorted = (float4 *)(ws + L.sorted);
    double *records = (double *)(ws + L.records);
    double *sums = (double *)(ws + L.sums);

    int alt_offered = 0;
    for (int i = 0; i < nch; ++i) if (ch[i].alt_gate == 1) alt_offered = 1;
    const int hint_class = hint_class_of(flags);
    int hint_pieces = hint_pieces_of(flags);
    // no hint, automatic: tell the setup kernel which centred-form launch is on offer for a uniform grid with a general start
    if (hint_class == -3 && is_auto)
        for (int i = 0; i < nch; ++i) if (ch[i].variant == V_CENT) hint_pieces = (ch[i].n_chunks << 8) | (ch[i].K / 8);
    if (hint_class == 0 && nch == 1 && ch[0].variant == V_RECUR) {
        // hinted q[0] == 0 and a single recurrence launch: it is the one sized for M - 1 indices exactly when that pays
        Choice c2[2];
        alt_offered = (recur_choices(c2, M) == 2) ? 1 : 0;
    }
    const bool pack_here = !pre && (int64_t)N * B <= DEBYE_PACK_IN_SETUP;      // small inputs: the setup CTA gathers too
    // tile split over GPUs: the pairs CTAs of the other ranks do not run here; their records must read as zero
    if (shard_world > 1) CU(cudaMemsetAsync(records, 0, L.sums - L.records, stream));
    if (!pre) debye::debye_setup_kernel<<<1, DEBYE_SETUP_THREADS, 0, stream>>>(plan, type, q, perm, N, T, M, B, alt_offered, hint_class, hint_pieces, xyz, sorted, pack_here ? 1 : 0, weight,
                                                                                shard_rank, shard_world);
    if (!pack_here) {
        int64_t total = (int64_t)N * B;
        int blocks = (int)((total + 255) / 256);
        if (blocks > sms * 16) blocks = sms * 16;
        // with a plan the pack kernel is the first kernel of the call: an ordinary launch (its pdl_wait returns at once)
        if (pre) debye::debye_pack_kernel<<<blocks, 256, 0, stream>>>(plan, xyz, type, perm, sorted, N, B, weight);
        else CU(launch_pdl(debye::debye_pack_kernel, dim3(blocks), dim3(256), stream, (const DevPlan *)plan, xyz, type, (const int32_t *)perm, sorted, N, B, weight));
    }
    if (weight) CU(launch_pdl(debye::debye_weight_sums_kernel, dim3(T), dim3(32), stream, plan, (const float4 *)sorted));
    if (ev0) CU(cudaEventRecord(ev0, stream));
    for (int i = 0; i < nch; ++i) {
        debye_pairs_fn fn = debye_get_pairs_kernel(ch[i].variant, ch[i].K, weight != nullptr, shard_world > 1);
        if (!fn) return DEBYE_EUNSUPPORTED;
        // slow-path threshold on theta = r * (smallest grid step or smallest |q|): see DESIGN.md section 6
        const float theta_min = (ch[i].variant == V_RECUR) ? 0.002f : 0.004f;
        CU(launch_pdl(fn, dim3(G[i]), dim3(DEBYE_IB), stream, (const DevPlan *)plan, (const float4 *)sorted, q, records, ch[i].n_chunks, is_auto, theta_min, ch[i].alt_gate));
    }
    if (ev1) CU(cudaEventRecord(ev1, stream));
    {
        // the final kernels repeat the device-side decisions of the pairs launches to find the one that did the work
        debye::FinalSets sets; sets.n = nch;
        int64_t red_blocks = 0;
        for (int i = 0; i < MAX_CHOICES; ++i) {
            const int j = i < nch ? i : 0;
            sets.s[i].variant = ch[j].variant; sets.s[i].K = ch[j].K; sets.s[i].n_chunks = ch[j].n_chunks; sets.s[i].G = G[j]; sets.s[i].alt_gate = ch[j].alt_gate;
            const int64_t nb = (int64_t)B * (T * (T + 1) / 2) * ch[j].n_chunks * ((ch[j].K + 31) / 32);
            if (nb > red_blocks) red_blocks = nb;
        }
        if (red_blocks > 0x7fffffff) return DEBYE_EUNSUPPORTED;
        CU(launch_pdl(debye::debye_reduce_kernel, dim3((unsigned)red_blocks), dim3(DEBYE_RED_THREADS), stream, (const DevPlan *)plan, (const double *)records, sums, is_auto, sets));
        const int blocks = B * ((M + DEBYE_FINAL_Q - 1) / DEBYE_FINAL_Q);
        CU(launch_pdl(debye::debye_epilogue_kernel, dim3(blocks), dim3(DEBYE_FINAL_THREADS), stream, (const DevPlan *)plan, (const double *)sums, fftab, q, out, is_auto, sets, mode));
    }
    if (mode == 1 && n_out) CU(cudaMemcpyAsync(n_out, plan->n_a, sizeof(int32_t) * T, cudaMemcpyDeviceToDevice, stream));
    CU(scratch_release(*order, stream));
    CU(cudaGetLastError());
    return DEBYE_OK;
}

int run_host(const float *xyz, const int32_t *type, int N, int B, const float *fftab, int T, const float *q, int M, double *out, uint32_t flags,
             cudaStream_t stream, const float *weight = nullptr)
{
    int st = validate(xyz, type, N, B, fftab, T, q, M, out, flags);
    if (st) return st;
    DevState *ds;
    char *base, *hbase = nullptr;
    size_t o_xyz, o_type, o_tab, o_q, o_out, o_w, o_in, total;
    {
        size_t o = 0;                              // the inputs first, contiguous, so that they can travel as one copy
        o_xyz = o; o += align_up((size_t)N * B * 12);
        o_type = o; o += align_up((size_t)N * 4);
        o_tab = o; o += align_up((size_t)T * M * 4);
        o_q = o; o += align_up((size_t)M * 4);
        o_w = o; o += align_up((size_t)N * 4);
        o_in = o;
        o_out = o; o += align_up((size_t)B * M * 8);
        total = o;
    }
    // Small inputs (for small proteins the transfers, not the pairs, dominate): gathered into a pinned staging buffer
    // on the host and copied ONCE instead of four or five copies of a few KB each.  One such call at a time per process: the
    // buffer is refilled by the next call, so the lock is held until this call's copy has been consumed (the final synchronise).
    const bool one_copy = o_in <= HOST_ONE_COPY_MAX;
    std::unique_lock<std::mutex> hlock(g_hstage_mu, std::defer_lock);
    if (one_copy) hlock.lock();
    {
        std::lock_guard<std::mutex> lock(g_mu);
        if ((st = dev_state(&ds))) return st;
        if ((st = ensure(&ds->stage, &ds->stage_bytes, total))) return st;
        base = (char *)ds->stage;
        if (one_copy) {
            if (ds->hstage_bytes < o_in) {
                if (ds->hstage) { CU(cudaFreeHost(ds->hstage)); ds->hstage = nullptr; ds->hstage_bytes = 0; }
                cudaError_t e = cudaHostAlloc(&ds->hstage, HOST_ONE_COPY_MAX, cudaHostAllocDefault);
                if (e != cudaSuccess) { (void)cudaGetLastError(); g_last_cuda = (int)e; ds->hstage = nullptr; return DEBYE_ENOMEM; }
                ds->hstage_bytes = HOST_ONE_COPY_MAX;
                if (!g_atexit) { g_atexit = true; atexit(shutdown_all); }
            }
            hbase = (char *)ds->hstage;
        }
        CU(scratch_acquire(ds->order, stream));    // the staging buffer is shared scratch too; run() releases behind the last kernel
    }
    if (one_copy) {
        memcpy(hbase + o_xyz, xyz, (size_t)N * B * 12);
        memcpy(hbase + o_type, type, (size_t)N * 4);
        memcpy(hbase + o_tab, fftab, (size_t)T * M * 4);
        memcpy(hbase + o_q, q, (size_t)M * 4);
        if (weight) memcpy(hbase + o_w, weight, (size_t)N * 4);
        CU(cudaMemcpyAsync(base, hbase, weight ? o_in : o_w, cudaMemcpyHostToDevice, stream));
    } else {
        CU(cudaMemcpyAsync(base + o_xyz, xyz, (size_t)N * B * 12, cudaMemcpyHostToDevice, stream));
        CU(cudaMemcpyAsync(base + o_type, type, (size_t)N * 4, cudaMemcpyHostToDevice, stream));
        CU(cudaMemcpyAsync(base + o_tab, fftab, (size_t)T * M * 4, cudaMemcpyHostToDevice, stream));
        CU(cudaMemcpyAsync(base + o_q, q, (size_t)M * 4, cudaMemcpyHostToDevice, stream));
        if (weight) CU(cudaMemcpyAsync(base + o_w, weight, (size_t)N * 4, cudaMemcpyHostToDevice, stream));
    }
    st = run((const float *)(base + o_xyz), (const int32_t *)(base + o_type), N, B, (const float *)(base + o_tab), T, (const float *)(base + o_q), M,
             (double *)(base + o_out), nullptr, flags, stream, 0, weight ? (const float *)(base + o_w) : nullptr);
    if (st) { if (one_copy) (void)cudaStreamSynchronize(stream); return st; }      // the pinned staging buffer must be drained before it is released
    CU(cudaMemcpyAsync(out, base + o_out, (size_t)B * M * 8, cudaMemcpyDeviceToHost, stream));
    CU(cudaStreamSynchronize(stream));             // the staging buffer is free again when this returns
    return DEBYE_OK;
}

}  // namespace

extern "C" {

int debye_profile(const float *xyz, const int32_t *type, int32_t N, const float *fftab, int32_t T, const float *q, int32_t M, double *I_out, uint32_t flags,
                  debye_stream_t stream)
{
    return run(xyz, type, N, 1, fftab, T, q, M, I_out, nullptr, flags, (cudaStream_t)stream, 0);
}

int debye_profile_batch(const float *xyz, const int32_t *type, int32_t N, int32_t B, const float *fftab, int32_t T, const float *q, int32_t M, double *I_out,
                        uint32_t flags, debye_stream_t stream)
{
    return run(xyz, type, N, B, fftab, T, q, M, I_out, nullptr, flags, (cudaStream_t)stream, 0);
}

int debye_profile_host(const float *xyz, const int32_t *type, int32_t N, const float *fftab, int32_t T, const float *q, int32_t M, double *I_out, uint32_t flags,
                       debye_stream_t stream)
{
    return run_host(xyz, type, N, 1, fftab, T, q, M, I_out, flags, (cudaStream_t)stream);
}

int debye_profile_batch_host(const float *xyz, const int32_t *type, int32_t N, int32_t B, const float *fftab, int32_t T, const float *q, int32_t M,
                             double *I_out, uint32_t flags, debye_stream_t stream)
{
    return run_host(xyz, type, N, B, fftab, T, q, M, I_out, flags, (cudaStream_t)stream);
}

int debye_profile_weighted(const float *xyz, const int32_t *type, const float *weight, int32_t N, const float *fftab, int32_t T, const float *q, int32_t M,
                           double *I_out, uint32_t flags, debye_stream_t stream)
{
    if (!weight) return DEBYE_EINVAL;
    return run(xyz, type, N, 1, fftab, T, q, M, I_out, nullptr, flags, (cudaStream_t)stream, 0, weight);
}

int debye_profile_batch_weighted(const float *xyz, const int32_t *type, const float *weight, int32_t N, int32_t B, const float *fftab, int32_t T, const float *q,
                                 int32_t M, double *I_out, uint32_t flags, debye_stream_t stream)
{
    if (!weight) return DEBYE_EINVAL;
    return run(xyz, type, N, B, fftab, T, q, M, I_out, nullptr, flags, (cudaStream_t)stream, 0, weight);
}

int debye_profile_weighted_host(const float *xyz, const int32_t *type, const float *weight, int32_t N, const float *fftab, int32_t T, const float *q, int32_t M,
                                double *I_out, uint32_t flags, debye_stream_t stream)
{
    if (!weight) return DEBYE_EINVAL;
    return run_host(xyz, type, N, 1, fftab, T, q, M, I_out, flags, (cudaStream_t)stream, weight);
}

int debye_partials(const float *xyz, const int32_t *type, int32_t N, int32_t B, const float *q, int32_t T, int32_t M, double *S_out, int32_t *n_out,
                   uint32_t flags, debye_stream_t stream)
{
    return run(xyz, type, N, B, nullptr, T, q, M, S_out, n_out, flags, (cudaStream_t)stream, 1);
}

int debye_partials_shard(const float *xyz, const int32_t *type, int32_t N, int32_t B, const float *q, int32_t T, int32_t M, double *S_out, int32_t *n_out,
                         uint32_t flags, int32_t shard_rank, int32_t shard_world, debye_stream_t stream)
{
    if (shard_world < 1 || shard_world > 4096 || shard_rank < 0 || shard_rank >= shard_world) return DEBYE_EINVAL;
    return run(xyz, type, N, B, nullptr, T, q, M, S_out, n_out, flags, (cudaStream_t)stream, 1, nullptr, nullptr, shard_rank, shard_world);
}

int debye_profile_from_partials(const double *S_parts, int32_t n_parts, const int32_t *n_a, const float *fftab, int32_t B, int32_t T, int32_t M, double *I_out,
                                debye_stream_t stream)
{
    if (!S_parts || !n_a || !fftab || !I_out) return DEBYE_EINVAL;
    if (n_parts < 1 || n_parts > 4096 || B < 1 || B > 65535 || T < 1 || T > DEBYE_MAX_TYPES || M < 1 || M > DEBYE_MAX_Q) return DEBYE_EINVAL;
    debye::debye_combine_kernel<<<dim3((M + 127) / 128, B), 128, 0, (cudaStream_t)stream>>>(S_parts, n_parts, n_a, fftab, B, T, M, I_out);
    CU(cudaGetLastError());
    return DEBYE_OK;
}

namespace {
// per-atom form factors, recurrence (debye_peratom_recur.cuh): pack (+ grid check) | self terms | pairs | final.  Called with g_mu held.
// B conformers (xyz[B][N][3], I_out[B][M]) share the table: one unit line conformer -> chunk -> row -> j.
int run_peratom_recur(DevState *ds, const float *xyz, const float *ff, int N, const float *q, int M, double *I_out, int cls, int n_chunks, int K, cudaStream_t stream,
                      int B = 1)
{
    debye_peratom_recur_fn fn = debye_get_peratom_recur_kernel(K, B > 1);
    if (!fn) return DEBYE_EUNSUPPORTED;
    int st;
    const int rows = debye_diag_rows(N);
    const int64_t U = (rows > 0 ? debye_diag_row_prefix(N, rows) : 0) * n_chunks * B;
    const int64_t one_wave = (int64_t)ds->sms * (K <= 64 ? 3 : 2);
    int64_t G = U / DEBYE_PAR_UNITS_PER_CTA / one_wave * one_wave;                 // whole waves, at least ~150 units (j atoms x 128 i atoms) per CTA
    if (G > one_wave * 16) G = one_wave * 16;
    if (G < one_wave) { G = U / 8; if (G > one_wave) G = one_wave; }
    if (G < 1) G = 1;
    size_t o = 0;
    const size_t o_plan = o; o += align_up(sizeof(debye::PeratomPlan));
    const size_t o_pos = o; o += align_up((size_t)N * B * 16 + 16 * DEBYE_PAR_JT);
    const size_t o_ffp = o; o += align_up((size_t)n_chunks * N * K * 4 + (size_t)DEBYE_PAR_JT * K * 4);
    const size_t o_rec = o; o += align_up((size_t)(G + (int64_t)n_chunks * B) * K * 8);
    const size_t o_self = o; o += align_up((size_t)DEBYE_PA_SLICES * 2 * M * 8);
    char *ws;
    if (ds->user_ws) { if (ds->user_bytes < o) return DEBYE_ENOMEM; ws = (char *)ds->user_ws; }
    else { if ((st = ensure(&ds->ws, &ds->ws_bytes, o))) return st; ws = (char *)ds->ws; }
    debye::PeratomPlan *plan = (debye::PeratomPlan *)(ws + o_plan);
    float4 *pos4 = (float4 *)(ws + o_pos);
    float *ffp = (float *)(ws + o_ffp);
    double *records = (double *)(ws + o_rec), *selfbuf = (double *)(ws + o_self);
    CU(scratch_acquire(ds->order, stream));
    int pb = (int)((std::max((int64_t)N * K, (int64_t)N * B) + 255) / 256);
    if (pb > ds->sms * 8) pb = ds->sms * 8;
    if (pb < 1) pb = 1;
    debye::debye_peratom_pack_kernel<<<dim3(pb, n_chunks + 1), 256, 0, stream>>>(xyz, ff, q, N, M, K, n_chunks, cls, pos4, ffp, plan, B);
    // The rest of the chain with programmatic stream serialisation -- every kernel starts with pdl_wait() (debye_plan.cuh) --
    // which hides the launch gaps: 1000 atoms 48 -> 42 us per call, cfg2 0.827 -> 0.819 ms, cfg3 unchanged (measured on B200).
    const bool chain_pdl = DEBYE_PA_PDL != 0;
    if (chain_pdl) CU(launch_pdl(debye::debye_peratom_self_kernel, dim3((M + 31) / 32, DEBYE_PA_SLICES), dim3(256), stream, ff, N, M, selfbuf));
    else debye::debye_peratom_self_kernel<<<dim3((M + 31) / 32, DEBYE_PA_SLICES), 256, 0, stream>>>(ff, N, M, selfbuf);
    if (ds->ev0) CU(cudaEventRecord(ds->ev0, stream));
    if (U > 0) {
        if (chain_pdl) CU(launch_pdl(fn, dim3((unsigned)G), dim3(DEBYE_IB), stream, (const float4 *)pos4, (const float *)ffp, q, (const debye::PeratomPlan *)plan, N, M, n_chunks, 0.002f, records, B));
        else fn<<<(int)G, DEBYE_IB, 0, stream>>>(pos4, ffp, q, plan, N, M, n_chunks, 0.002f, records, B);
    }
    if (ds->ev1) CU(cudaEventRecord(ds->ev1, stream));
    if (chain_pdl) CU(launch_pdl(debye::debye_peratom_final_kernel, dim3((M + 31) / 32, B), dim3(32 * DEBYE_PA_FS), stream, (const double *)records, (const double *)selfbuf, q, N, M, n_chunks,
                                 (int)G, K, I_out, (const int32_t *)plan));
    else debye::debye_peratom_final_kernel<<<dim3((M + 31) / 32, B), 32 * DEBYE_PA_FS, 0, stream>>>(records, selfbuf, q, N, M, n_chunks, (int)G, K, I_out, (const int32_t *)plan);
    CU(scratch_release(ds->order, stream));
    CU(cudaGetLastError());
    return DEBYE_OK;
}
}  // namespace

namespace {
// per-atom form factors, one small structure, hinted one-chunk grid: ONE cooperative launch (debye_peratom_small.cuh).  Called with g_mu held.
int run_peratom_small(DevState *ds, const float *xyz, const float *ff, int N, const float *q, int M, double *I_out, int cls, int K, cudaStream_t stream)
{
    debye_peratom_small_fn fn = debye_get_peratom_small_kernel(K);
    if (!fn) return DEBYE_EUNSUPPORTED;
    int st;
    static bool attr_set[MAX_DEV][DEBYE_KMAX_F32 / 8 + 1];
    int dev = 0;
    CU(cudaGetDevice(&dev));
    if (!attr_set[dev][K / 8]) {
        CU(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)debye::debye_peratom_small_dyn_smem(DEBYE_PAS_NMAX, DEBYE_KMAX_F32)));
        attr_set[dev][K / 8] = true;
    }
    // cooperative launch: the grid is one resident wave, DEBYE_PAS_CTAS_PER_SM CTAs per SM at most (if that many fit); at least
    // ~DEBYE_PAS_UNITS units (j atom x 128 i atoms) per CTA
    int occ = 0;
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, DEBYE_IB, debye::debye_peratom_small_dyn_smem(N, K)));
    if (occ < 1) occ = 1;
    if (occ > DEBYE_PAS_CTAS_PER_SM) occ = DEBYE_PAS_CTAS_PER_SM;
    int64_t g = ((int64_t)N * N / (2 * DEBYE_IB) + 1) / DEBYE_PAS_UNITS;
    if (g > (int64_t)ds->sms * occ) g = (int64_t)ds->sms * occ;
    if (g > DEBYE_PAS_GMAX) g = DEBYE_PAS_GMAX;
    if (g < 1) g = 1;
    const int G = (int)g;
    const size_t need = align_up((size_t)G * K * 8);
    char *ws;
    if (ds->user_ws) { if (ds->user_bytes < need) return DEBYE_ENOMEM; ws = (char *)ds->user_ws; }
    else { if ((st = ensure(&ds->ws, &ds->ws_bytes, need))) return st; ws = (char *)ds->ws; }
    double *records = (double *)ws;
    CU(scratch_acquire(ds->order, stream));
    if (ds->ev0) CU(cudaEventRecord(ds->ev0, stream));
    int hc = cls;
    void *args[] = {(void *)&xyz, (void *)&ff, (void *)&q, (void *)&N, (void *)&M, (void *)&hc, (void *)&records, (void *)&I_out};
    CU(cudaLaunchCooperativeKernel((const void *)fn, dim3(G), dim3(DEBYE_IB), args, debye::debye_peratom_small_dyn_smem(N, K), stream));
    if (ds->ev1) CU(cudaEventRecord(ds->ev1, stream));
    CU(scratch_release(ds->order, stream));
    CU(cudaGetLastError());
    return DEBYE_OK;
}
}  // namespace

int debye_profile_peratom(const float *xyz, const float *ff, int32_t N, const float *q, int32_t M, double *I_out, uint32_t flags, debye_stream_t stream_)
{
    cudaStream_t stream = (cudaStream_t)stream_;
    if (!xyz || !ff || !q || !I_out) return DEBYE_EINVAL;
    if (N < 1 || M < 1 || M > DEBYE_MAX_Q) return DEBYE_EINVAL;
    // FP64, FP32 with one MUFU.SIN per term (DEBYE_SINC_MUFU, or any grid without a hint), or -- with a grid hint that promises
    // q_k = (k + koff) dq -- the recurrence (DEBYE_SINC_RECUR or automatic)
    // (a piecewise-uniform hint, which debye_q_hint may return, is accepted and means "no uniform grid" here)
    const uint32_t hint_bits = DEBYE_QHINT | DEBYE_QHINT_UNIFORM | DEBYE_QHINT_START0 | DEBYE_QHINT_STARTDQ | DEBYE_QHINT_PIECES |
                               (31u << DEBYE_QHINT_NPIECES_SHIFT) | (31u << DEBYE_QHINT_PIECEK_SHIFT);
    if (flags & ~(uint32_t)(DEBYE_FP64 | DEBYE_SINC_MUFU | DEBYE_SINC_RECUR | hint_bits)) return DEBYE_EINVAL;
    if ((flags & DEBYE_FP64) && (flags & (DEBYE_SINC_MUFU | DEBYE_SINC_RECUR))) return DEBYE_EINVAL;
    if ((flags & DEBYE_SINC_MUFU) && (flags & DEBYE_SINC_RECUR)) return DEBYE_EINVAL;
    {
        const uint32_t sub = flags & (DEBYE_QHINT_UNIFORM | DEBYE_QHINT_START0 | DEBYE_QHINT_STARTDQ), st2 = flags & (DEBYE_QHINT_START0 | DEBYE_QHINT_STARTDQ);
        if ((sub && !(flags & DEBYE_QHINT)) || (st2 && !(flags & DEBYE_QHINT_UNIFORM)) || st2 == (DEBYE_QHINT_START0 | DEBYE_QHINT_STARTDQ)) return DEBYE_EINVAL;
    }
    if (N > (1 << 24)) return DEBYE_EUNSUPPORTED;
    const bool f64 = (flags & DEBYE_FP64) != 0;
    if (flags & DEBYE_SINC_RECUR) {        // the recurrence was demanded: only for a hinted grid q_k = (k + koff) dq of at most 2 chunks
        const int cls = hint_class_of(flags);
        if ((cls != 0 && cls != 1) || M - (cls == 0 ? 1 : 0) < 1 || choose(V_RECUR, M - (cls == 0 ? 1 : 0)).n_chunks > 2) return DEBYE_EUNSUPPORTED;
    }
    std::lock_guard<std::mutex> lock(g_mu);
    DevState *ds; int st;
    if ((st = dev_state(&ds))) return st;
    {   // the recurrence: hinted grid q_k = (k + koff) dq, at most two chunks of 128 chain indices
        const int cls = hint_class_of(flags);
        const int n_idx = M - (cls == 0 ? 1 : 0);
        if (!f64 && !(flags & DEBYE_SINC_MUFU) && (cls == 0 || cls == 1) && n_idx >= 1) {
            const Choice c = choose(V_RECUR, n_idx);
            // one small structure on a one-chunk grid: a single fused launch (debye_peratom_small.cuh)
            if (c.n_chunks == 1 && N <= DEBYE_PAS_NMAX) return run_peratom_small(ds, xyz, ff, N, q, M, I_out, cls, (c.K + 7) / 8 * 8, stream);
            if (c.n_chunks <= 2) return run_peratom_recur(ds, xyz, ff, N, q, M, I_out, cls, c.n_chunks, (c.K + 7) / 8 * 8, stream);
        }
    }
    const int KQ = debye::debye_peratom_kq(M);
    const int n_chunks = (M + KQ - 1) / KQ;
    const int rows = debye_diag_rows(N);
    const int64_t U = (rows > 0 ? debye_diag_row_prefix(N, rows) : 0) * n_chunks;
    // resident CTAs x up to 8 waves, at least ~192 units (j atoms x 128 i atoms x 32 q) per CTA
    // whole waves of resident CTAs (a grid slightly above one wave runs its last CTAs alone: N = 4 000 took 0.25 ms with
    // 594 CTAs, 0.20 ms with 589); small structures: one full wave of short ranges (at least 24 units each)
    const int64_t one_wave = (int64_t)ds->sms * (f64 ? 2 : DEBYE_PA_CTAS);
    const int64_t Gmax = one_wave * 8;
    int64_t G = U / (192 * DEBYE_PA_KQ / KQ);
    if (G < one_wave) { G = U / 24; if (G > one_wave) G = one_wave; }
    else G = G / one_wave * one_wave;
    if (G > Gmax) G = Gmax;
    if (G < 1) G = 1;
    size_t o = 0;
    const size_t o_rec = o; o += align_up((size_t)(G + n_chunks) * DEBYE_PA_KQ * 8);
    const size_t o_self = o; o += align_up((size_t)DEBYE_PA_SLICES * 2 * M * 8);
    char *ws;
    if (ds->user_ws) { if (ds->user_bytes < o) return DEBYE_ENOMEM; ws = (char *)ds->user_ws; }
    else { if ((st = ensure(&ds->ws, &ds->ws_bytes, o))) return st; ws = (char *)ds->ws; }
    double *records = (double *)(ws + o_rec), *selfbuf = (double *)(ws + o_self);
    CU(scratch_acquire(ds->order, stream));
    const bool chain_pdl = DEBYE_PA_PDL != 0;  // programmatic stream serialisation along the chain (as run_peratom_recur)
    debye::debye_peratom_self_kernel<<<dim3((M + 31) / 32, DEBYE_PA_SLICES), 256, 0, stream>>>(ff, N, M, selfbuf);
    if (ds->ev0) CU(cudaEventRecord(ds->ev0, stream));
    if (U > 0) {
#define DEBYE_PA_LAUNCH(KQ_)                                                                                                              \
    case KQ_:                                                                                                                           \
        if (f64) { if (chain_pdl) CU(launch_pdl(debye::debye_peratom_pairs_kernel<true, KQ_>, dim3((unsigned)G), dim3(DEBYE_IB), stream, xyz, ff, q, N, M, n_chunks, records));    \
                   else debye::debye_peratom_pairs_kernel<true, KQ_><<<(int)G, DEBYE_IB, 0, stream>>>(xyz, ff, q, N, M, n_chunks, records); }                                 \
        else { if (chain_pdl) CU(launch_pdl(debye::debye_peratom_pairs_kernel<false, KQ_>, dim3((unsigned)G), dim3(DEBYE_IB), stream, xyz, ff, q, N, M, n_chunks, records));      \
               else debye::debye_peratom_pairs_kernel<false, KQ_><<<(int)G, DEBYE_IB, 0, stream>>>(xyz, ff, q, N, M, n_chunks, records); }                                   \
        break;
        switch (KQ) { DEBYE_PA_LAUNCH(16) DEBYE_PA_LAUNCH(20) DEBYE_PA_LAUNCH(24) DEBYE_PA_LAUNCH(28) DEBYE_PA_LAUNCH(32) default: return DEBYE_EUNSUPPORTED; }
#undef DEBYE_PA_LAUNCH
    }
    if (ds->ev1) CU(cudaEventRecord(ds->ev1, stream));
    if (chain_pdl) CU(launch_pdl(debye::debye_peratom_final_kernel, dim3((M + 31) / 32), dim3(32 * DEBYE_PA_FS), stream, (const double *)records, (const double *)selfbuf, q, N, M, n_chunks,
                                 (int)G, KQ, I_out, (const int32_t *)nullptr));
    else debye::debye_peratom_final_kernel<<<(M + 31) / 32, 32 * DEBYE_PA_FS, 0, stream>>>(records, selfbuf, q, N, M, n_chunks, (int)G, KQ, I_out, nullptr);
    CU(scratch_release(ds->order, stream));
    CU(cudaGetLastError());
    return DEBYE_OK;
}

int debye_profile_peratom_batch(const float *xyz, const float *ff, int32_t N, int32_t B, const float *q, int32_t M, double *I_out, uint32_t flags, debye_stream_t stream_)
{
    if (B < 1 || B > 65535) return DEBYE_EINVAL;                      // the final kernel puts the conformer on blockIdx.y
    if (B == 1) return debye_profile_peratom(xyz, ff, N, q, M, I_out, flags, stream_);
    if (!xyz || !ff || !q || !I_out || N < 1 || M < 1 || M > DEBYE_MAX_Q) return DEBYE_EINVAL;
    if ((int64_t)N * B > ((int64_t)1 << 31)) return DEBYE_EUNSUPPORTED;
    // hinted grid q_k = (k + koff) dq: ONE launch sequence for all conformers (the recurrence; the table is packed once)
    const int cls = hint_class_of(flags);
    const int n_idx = M - (cls == 0 ? 1 : 0);
    const bool other = (flags & (DEBYE_FP64 | DEBYE_SINC_MUFU)) != 0;
    if (!other && (cls == 0 || cls == 1) && n_idx >= 1 && choose(V_RECUR, n_idx).n_chunks <= 2) {
        // argument checks of the single-structure entry (flags, sizes) on the first conformer's terms
        const uint32_t hint_bits = DEBYE_QHINT | DEBYE_QHINT_UNIFORM | DEBYE_QHINT_START0 | DEBYE_QHINT_STARTDQ;
        if (flags & ~(uint32_t)(DEBYE_SINC_RECUR | hint_bits)) return DEBYE_EINVAL;
        if ((flags & DEBYE_QHINT_START0) && (flags & DEBYE_QHINT_STARTDQ)) return DEBYE_EINVAL;
        if (N > (1 << 24)) return DEBYE_EUNSUPPORTED;
        std::lock_guard<std::mutex> lock(g_mu);
        DevState *ds; int st;
        if ((st = dev_state(&ds))) return st;
        const Choice c = choose(V_RECUR, n_idx);
        return run_peratom_recur(ds, xyz, ff, N, q, M, I_out, cls, c.n_chunks, (c.K + 7) / 8 * 8, (cudaStream_t)stream_, B);
    }
    // any other grid or variant: the single-structure sequence per conformer on the same stream (stream order serialises the
    // shared scratch)
    for (int b = 0; b < B; ++b) {
        const int st = debye_profile_peratom(xyz + (size_t)b * N * 3, ff, N, q, M, I_out + (size_t)b * M, flags, stream_);
        if (st) return st;
    }
    return DEBYE_OK;
}

int debye_profile_peratom_host(const float *xyz, const float *ff, int32_t N, const float *q, int32_t M, double *I_out, uint32_t flags, debye_stream_t stream_)
{
    cudaStream_t stream = (cudaStream_t)stream_;
    if (!xyz || !ff || !q || !I_out) return DEBYE_EINVAL;
    if (N < 1 || M < 1 || M > DEBYE_MAX_Q) return DEBYE_EINVAL;
    if (N > (1 << 24)) return DEBYE_EUNSUPPORTED;
    DevState *ds; int st; char *base;
    size_t o = 0;
    const size_t o_xyz = o; o += align_up((size_t)N * 12);
    const size_t o_ff = o; o += align_up((size_t)N * M * 4);
    const size_t o_q = o; o += align_up((size_t)M * 4);
    const size_t o_out = o; o += align_up((size_t)M * 8);
    {
        std::lock_guard<std::mutex> lock(g_mu);
        if ((st = dev_state(&ds))) return st;
        if ((st = ensure(&ds->stage, &ds->stage_bytes, o))) return st;
        base = (char *)ds->stage;
        CU(scratch_acquire(ds->order, stream));
    }
    CU(cudaMemcpyAsync(base + o_xyz, xyz, (size_t)N * 12, cudaMemcpyHostToDevice, stream));
    CU(cudaMemcpyAsync(base + o_ff, ff, (size_t)N * M * 4, cudaMemcpyHostToDevice, stream));
    CU(cudaMemcpyAsync(base + o_q, q, (size_t)M * 4, cudaMemcpyHostToDevice, stream));
    st = debye_profile_peratom((const float *)(base + o_xyz), (const float *)(base + o_ff), N, (const float *)(base + o_q), M, (double *)(base + o_out), flags, stream_);
    if (st) return st;
    CU(cudaMemcpyAsync(I_out, base + o_out, (size_t)M * 8, cudaMemcpyDeviceToHost, stream));
    CU(cudaStreamSynchronize(stream));
    return DEBYE_OK;
}

int debye_plan_create(debye_plan **out, const int32_t *type, int32_t N, int32_t B, int32_t T, const float *q, int32_t M, const float *weight, uint32_t flags,
                      debye_stream_t stream_)
{
    static const char dummy = 0;
    cudaStream_t stream = (cudaStream_t)stream_;
    if (!out) return DEBYE_EINVAL;
    *out = nullptr;
    int st = validate(&dummy, type, N, B, &dummy, T, q, M, &dummy, flags);
    if (st) return st;
    debye_plan *p = new debye_plan();
    p->N = N; p->B = B; p->T = T; p->M = M; p->flags = flags; p->buf = nullptr; p->ws = nullptr; p->ws_bytes = 0;
    auto fail = [&](int code) { if (p->buf) cudaFree(p->buf); delete p; return code; };
    if (cudaGetDevice(&p->device) != cudaSuccess) return fail(DEBYE_ECUDA);
    const uint32_t all_hint_bits = DEBYE_QHINT | DEBYE_QHINT_UNIFORM | DEBYE_QHINT_START0 | DEBYE_QHINT_STARTDQ | DEBYE_QHINT_PIECES |
                                   (31u << DEBYE_QHINT_NPIECES_SHIFT) | (31u << DEBYE_QHINT_PIECEK_SHIFT);
    // a piecewise-uniform grid (the centred product form) is recognised on a host copy of q: the launch is sized from its pieces
    uint32_t pieces_hint = 0;
    {
        std::vector<float> qh((size_t)M);
        if (cudaMemcpyAsync(qh.data(), q, (size_t)M * 4, cudaMemcpyDeviceToHost, stream) != cudaSuccess) return fail(DEBYE_ECUDA);
        if (cudaStreamSynchronize(stream) != cudaSuccess) return fail(DEBYE_ECUDA);
        const uint32_t hh = debye_q_hint(qh.data(), M);
        if (hh & DEBYE_QHINT_PIECES) pieces_hint = hh;
    }
    if ((flags & DEBYE_SINC_CENTRED) && !pieces_hint) return fail(DEBYE_EUNSUPPORTED);
    size_t o = 0;
    const size_t o_plan = o; o += align_up(sizeof(DevPlan));
    const size_t o_perm = o; o += align_up((size_t)N * 4);
    const size_t o_q = o; o += align_up((size_t)M * 4);
    const size_t o_w = o; o += align_up((size_t)N * 4);
    const size_t o_t = o; o += align_up((size_t)N * 4);
    const size_t o_ws = o;
    {   // the plan's own scratch, sized for any grid class the setup step may find (the hint is resolved below)
        size_t need = 0;
        const uint32_t base_flags = flags & ~all_hint_bits;
        if (pieces_hint) need = debye_workspace_bytes(N, B, T, M, base_flags | pieces_hint);
        const uint32_t hints[4] = {DEBYE_QHINT, DEBYE_QHINT | DEBYE_QHINT_UNIFORM, DEBYE_QHINT | DEBYE_QHINT_UNIFORM | DEBYE_QHINT_START0,
                                   DEBYE_QHINT | DEBYE_QHINT_UNIFORM | DEBYE_QHINT_STARTDQ};
        for (int i = 0; i < 4; ++i) { const size_t b = debye_workspace_bytes(N, B, T, M, base_flags | hints[i]); if (b > need) need = b; }
        if (need == 0) return fail(DEBYE_EINVAL);
        p->ws_bytes = need; o += align_up(need);
    }
    if (cudaMalloc((void **)&p->buf, o) != cudaSuccess) { (void)cudaGetLastError(); p->buf = nullptr; return fail(DEBYE_ENOMEM); }
    p->plan = (DevPlan *)(p->buf + o_plan); p->perm = (int32_t *)(p->buf + o_perm); p->q = (float *)(p->buf + o_q);
    p->weight = weight ? (float *)(p->buf + o_w) : nullptr;
    p->ws = p->buf + o_ws;
    p->type = (int32_t *)(p->buf + o_t);          // small structures re-sort per call inside the one fused launch
    if (cudaMemcpyAsync(p->type, type, (size_t)N * 4, cudaMemcpyDeviceToDevice, stream) != cudaSuccess) return fail(DEBYE_ECUDA);
    if (cudaMemcpyAsync(p->q, q, (size_t)M * 4, cudaMemcpyDeviceToDevice, stream) != cudaSuccess) return fail(DEBYE_ECUDA);
    if (weight && cudaMemcpyAsync(p->weight, weight, (size_t)N * 4, cudaMemcpyDeviceToDevice, stream) != cudaSuccess) return fail(DEBYE_ECUDA);
    // the setup step, once; then read its verdict on the grid back (the only synchronisation of the plan's life)
    debye::debye_setup_kernel<<<1, DEBYE_SETUP_THREADS, 0, stream>>>(p->plan, type, p->q, p->perm, N, T, M, B, 1, pieces_hint ? -4 : -3, hint_pieces_of(pieces_hint), nullptr, nullptr, 0,
                                                                     p->weight, 0, 1);
    DevPlan head;
    if (cudaMemcpyAsync(&head, p->plan, offsetof(DevPlan, seg_off), cudaMemcpyDeviceToHost, stream) != cudaSuccess) return fail(DEBYE_ECUDA);
    if (cudaStreamSynchronize(stream) != cudaSuccess) return fail(DEBYE_ECUDA);
    uint32_t hint = DEBYE_QHINT;
    if (head.uniform) hint |= DEBYE_QHINT_UNIFORM;
    if (head.uniform && head.zero_start == 0) hint |= DEBYE_QHINT_START0;
    if (head.uniform && head.zero_start == 1) hint |= DEBYE_QHINT_STARTDQ;
    if (pieces_hint) hint = pieces_hint;
    p->flags = (flags & ~all_hint_bits) | hint;
    *out = p;
    return DEBYE_OK;
}

int debye_plan_execute(debye_plan *p, const float *xyz, const float *fftab, double *I_out, debye_stream_t stream)
{
    static const int32_t dummy_type = 0;
    if (!p) return DEBYE_EINVAL;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != p->device) return DEBYE_EINVAL;
    return run(xyz, &dummy_type, p->N, p->B, fftab, p->T, p->q, p->M, I_out, nullptr, p->flags, (cudaStream_t)stream, 0, p->weight, p);
}

void debye_plan_destroy(debye_plan *p)
{
    if (!p) return;
    if (p->buf) cudaFree(p->buf);
    if (p->order.done) cudaEventDestroy(p->order.done);
    delete p;
}

uint32_t debye_q_hint(const float *q_host, int32_t M)
{
    if (!q_host || M < 1) return 0;
    const double q0 = (double)q_host[0];
    const double dq = debye_grid_dq(q0, (double)q_host[M - 1], M);
    float dev = 0.f, qmax = 0.f;
    for (int k = 0; k < M; ++k) {
        const float d = debye_grid_dev((double)q_host[k], k, q0, dq), a = fabsf(q_host[k]);
        if (d > dev) dev = d;
        if (a > qmax) qmax = a;
    }
    const int cls = debye_grid_class(q0, dq, dev, qmax);
    // a uniform grid from 0 or dq with more than 256 chain indices would need more than two residue-class chunks, for which the
    // recurrence only has its chain form (2 lane-operations per term): contiguous pieces of the centred form are twice as fast
    // (measured, 30 000 atoms x 1000 q: 6.5 -> 15.7 T pair.q/s; 3 000 atoms x 512 q: 5.9 -> 9.7 T)
    const bool many_chunks = cls >= 0 && M - (cls == 0 ? 1 : 0) > 2 * DEBYE_KMAX_F32;
    if (cls == -2 || (cls == -1 && DEBYE_CENT_FOR_GENERAL_START) || many_chunks) {
        // not one uniform grid from 0 or dq: a few uniform pieces (the centred product form) if the grid has that shape
        // ... and if it pays: a piece costs its start-up (~110 issue cycles per pair) plus one packed lane per accumulator, the MUFU
        // kernel 8 cycles per q -- a grid of many short pieces (any 40 random points are 20 "uniform" pieces of two) stays there
        const uint32_t fp = debye_q_hint_pieces(q_host, M);
        if (fp) {
            const int64_t np = ((fp >> DEBYE_QHINT_NPIECES_SHIFT) & 31u) + 1, Kp = 8 * (((fp >> DEBYE_QHINT_PIECEK_SHIFT) & 31u) + 1);
            if (np == 1 || np * (110 + Kp) < 8 * (int64_t)M) return fp;
        }
    }
    uint32_t f = DEBYE_QHINT;
    if (cls != -2) f |= DEBYE_QHINT_UNIFORM;
    if (cls == 0) f |= DEBYE_QHINT_START0;
    if (cls == 1) f |= DEBYE_QHINT_STARTDQ;
    return f;
}

uint32_t debye_q_hint_pieces(const float *q_host, int32_t M)
{
    if (!q_host || M < 1) return 0;
    DebyePieces P;
    if (!debye_find_pieces(q_host, M, P)) return 0;
    return DEBYE_QHINT | DEBYE_QHINT_PIECES | ((uint32_t)(P.n - 1) << DEBYE_QHINT_NPIECES_SHIFT) | ((uint32_t)(P.K / 8 - 1) << DEBYE_QHINT_PIECEK_SHIFT);
}

size_t debye_workspace_bytes(int32_t N, int32_t B, int32_t T, int32_t M, uint32_t flags)
{
    static const char dummy = 0;
    if (validate(&dummy, &dummy, N, B, &dummy, T, &dummy, M, &dummy, flags)) return 0;
    if (small_eligible(N, B, T, M, flags, nullptr, 1)) {
        std::lock_guard<std::mutex> lock(g_mu);
        DevState *ds; int G = 192 * 4;
        const int K = small_K(M, flags);
        if (dev_state(&ds) == DEBYE_OK) { int g = 0; if (small_grid(ds, N, T, K, &g) == DEBYE_OK) G = g; }
        (void)cudaGetLastError();
        return small_ws_bytes(T, K, G);
    }
    Choice ch[MAX_CHOICES]; int is_auto;
    int nch = variants_for(flags, ch, M, &is_auto);
    // exact when a CUDA device is current (same grid computation as the call itself; attribute queries only, no GPU work);
    // otherwise a safe upper bound: at most 192 SMs x 16 CTAs x 16 waves on any sm_100 part
    int Gmax = 192 * 16 * 16;
    {
        std::lock_guard<std::mutex> lock(g_mu);
        DevState *ds;
        if (dev_state(&ds) == DEBYE_OK) {
            int g = 0, gm = 0;
            bool ok = true;
            for (int i = 0; i < nch && ok; ++i) { ok = grid_for(ds, ch[i], N, B, &g) == DEBYE_OK; if (g > gm) gm = g; }
            if (ok && gm > 0) Gmax = gm;
        }
        (void)cudaGetLastError();
    }
    return layout(N, B, T, M, Gmax, ch, nch).total;
}

int debye_set_workspace(void *dev_ptr, size_t bytes)
{
    std::lock_guard<std::mutex> lock(g_mu);
    DevState *ds; int st;
    if ((st = dev_state(&ds))) return st;
    if (dev_ptr && ((uintptr_t)dev_ptr & 255)) return DEBYE_EINVAL;
    ds->user_ws = dev_ptr; ds->user_bytes = dev_ptr ? bytes : 0;
    return DEBYE_OK;
}

int debye_set_pairs_events(void *start_event, void *stop_event)
{
    std::lock_guard<std::mutex> lock(g_mu);
    DevState *ds; int st;
    if ((st = dev_state(&ds))) return st;
    if ((start_event == nullptr) != (stop_event == nullptr)) return DEBYE_EINVAL;
    ds->ev0 = (cudaEvent_t)start_event; ds->ev1 = (cudaEvent_t)stop_event;
    return DEBYE_OK;
}

void debye_shutdown(void)
{
    std::lock_guard<std::mutex> lock(g_mu);
    shutdown_all();
}

int debye_launch_info(int32_t N, int32_t B, int32_t T, int32_t M, uint32_t flags, int32_t *n_launches, int32_t *pairs_grid, int32_t *q_chunk, int32_t *n_chunks)
{
    static const char dummy = 0;
    int st = validate(&dummy, &dummy, N, B, &dummy, T, &dummy, M, &dummy, flags);
    if (st) return st;
    if (small_eligible(N, B, T, M, flags, nullptr, 1)) {      // one fused launch (debye_small.cuh)
        const int K = small_K(M, flags);
        if (n_launches) *n_launches = 1;
        if (q_chunk) *q_chunk = K;
        if (n_chunks) *n_chunks = 1;
        if (pairs_grid) {
            std::lock_guard<std::mutex> lock(g_mu);
            DevState *ds; int G = 0;
            if ((st = dev_state(&ds))) return st;
            if ((st = small_grid(ds, N, T, K, &G))) return st;
            *pairs_grid = G;
        }
        return DEBYE_OK;
    }
    Choice ch[MAX_CHOICES]; int is_auto;
    int nch = variants_for(flags, ch, M, &is_auto);
    const int lead = (nch > 1 && ch[0].alt_gate == 1) ? 1 : 0;     // report the launch sized for the general case
    if (n_launches) *n_launches = 3 + nch + (((int64_t)N * B <= DEBYE_PACK_IN_SETUP) ? 0 : 1);   // setup, [pack], pairs x nch, reduce, epilogue
    if (q_chunk) *q_chunk = ch[lead].K;
    if (n_chunks) *n_chunks = ch[lead].n_chunks;
    if (pairs_grid) {
        std::lock_guard<std::mutex> lock(g_mu);
        DevState *ds; int G = 0;
        if ((st = dev_state(&ds))) return st;
        if ((st = grid_for(ds, ch[lead], N, B, &G))) return st;
        *pairs_grid = G;
    }
    return DEBYE_OK;
}

const char *debye_strerror(int status)
{
    switch (status) {
        case DEBYE_OK: return "ok";
        case DEBYE_EINVAL: return "invalid argument";
        case DEBYE_EUNSUPPORTED: return "unsupported size";
        case DEBYE_ENOMEM: return "workspace allocation failed or supplied workspace too small";
        case DEBYE_ECUDA: return "CUDA runtime error (see debye_last_cuda_error)";
        default: return "unknown status";
    }
}

int debye_last_cuda_error(void) { return g_last_cuda; }
int debye_version(void) { return 100; }

}  // extern "C"
