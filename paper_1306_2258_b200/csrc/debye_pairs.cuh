// debye_pairs.cuh -- the all-pairs kernel of libdebye (steps S1-S6 of SURVEY.md section 8(a)).
//
// What one CTA does (PAPER.md:86-88 re-designed for sm_100a):
//   * owns a static contiguous range of "units" (one j atom x one row of 128 i atoms x K q-values), see
//     debye_plan.cuh; thread t keeps i atom t of the current row in registers (the paper's "private memory");
//   * streams the j atoms of the range through shared memory in 1 KB tiles with cp.async.bulk (TMA 1-D bulk
//     copy, SASS UBLKCP) completing on an mbarrier, double buffered (the paper's "local memory" blocks);
//   * because tiles are type-homogeneous, every pair of the range adds into the SAME K accumulators
//     S_ab(q_k) += sin(q_k r)/r  -- no form factor in the loop (north_star (c));
//   * FP32 accumulators are promoted to FP64 per flush: per-warp transpose through shared memory, each lane
//     sums 32 values in a fixed order, then a fixed-order sum over the 4 warps (north_star (f));
//   * per (conformer, type pair, q-chunk) the CTA writes one FP64 record; the final kernel adds records in
//     CTA order.
//
// Variants of the per-pair term evaluation (north_star (d), (e)):
//   V_RECUR    uniform grid q_k = qbase + k dq.  sin(q_k r) for all k of the chunk by the three-term
//              (Chebyshev) recurrence v_{k+S} = 2cos(S theta) v_k - v_{k-S}, theta = r dq, run as 4 packed
//              chains (8 residues mod S = 8 n_chunks) with fma.rn.f32x2 (SASS FFMA2) and accumulated with
//              add.rn.f32x2 (FADD2): 2 FP32-pipe lane-operations per term, no MUFU in the loop.  Start values
//              come from 4 (zero start) or 8 (general start) MUFU.SIN and a stride-4 bootstrap.
//   V_MUFU     any grid: explicit range reduction in turns (magic-number rounding, exact FMA remainder), one
//              MUFU.SIN per term.
//   V_ACCURATE any grid: libdevice sinf per term (reference variant).
//   V_F64      any grid: double differences, sqrt, libdevice sin; FP64 accumulators.
//   Pairs closer than r_cut (theta below the level where MUFU's absolute error matters) and coincident atoms
//   take a warp-uniform slow path: Taylor series of sinc for |x| < 0.25, sinf otherwise.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include "debye_plan.cuh"

typedef unsigned long long u64;

namespace debye {

// ---- packed f32x2 helpers (Blackwell FFMA2/FADD2) ----------------------------------------------------------
__device__ __forceinline__ u64 pk2(float lo, float hi) { u64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void upk2(u64 v, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { u64 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ u64 add2(u64 a, u64 b) { u64 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ u64 sub2(u64 a, u64 b) { u64 d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ float sin_mufu(float x) { float y; asm("sin.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rsqrt_mufu(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// sin(2 pi t) for t in turns, |t| < 2^22: magic-number round to nearest, exact remainder, MUFU.SIN
__device__ __forceinline__ float sin_turns(float t)
{
    const float MAGIC = 12582912.0f;             // 1.5 * 2^23
    float n = (t + MAGIC) - MAGIC;
    return sin_mufu((t - n) * 6.28318530717958648f);
}
// sin(2 pi r w) with the product's rounding error recovered by FMA (used where r*w can be hundreds of turns)
__device__ __forceinline__ float sin_turns_fma(float r, float w)
{
    const float MAGIC = 12582912.0f;
    float n = (fmaf(r, w, MAGIC)) - MAGIC;
    return sin_mufu(fmaf(r, w, -n) * 6.28318530717958648f);
}

// ---- accurate, UNBIASED trigonometry for the recurrence start-up ------------------------------------------------
// Measured on B200: MUFU.SIN has an absolute error of 3.4e-7 with a NON-ZERO MEAN (-1.1e-7 on
// (0, 0.5]).  A biased start value or a biased recurrence coefficient is a coherent phase / frequency error in every
// chain of every pair, and the cancellation in I(q) (condition number up to ~400 in cfg5) amplifies it to 7e-4.
// A relative frequency bias must stay below ~1e-9, so: frequencies are carried as hi + lo floats, the leading
// polynomial coefficient pi is split hi + lo, and everything else is round-to-nearest FMA arithmetic (unbiased).

// fractional part of r * (w + w_lo) in turns, in [-1/2, 1/2]: magic-number rounding, FMA remainders
__device__ __forceinline__ float reduce_turns(float r, float w, float w_lo)
{
    const float MAGIC = 12582912.0f;                 // 1.5 * 2^23
    const float n = fmaf(r, w, MAGIC) - MAGIC;
    return fmaf(r, w_lo, fmaf(r, w, -n));
}
// sh = sin(pi f), ch = cos(pi f) for |f| <= 1/2 (Taylor to pi^13/13! and pi^12/12!, remainders < 6e-9 / 4e-8)
__device__ __forceinline__ void sincos_pi(float f, float &sh, float &ch)
{
    const float y = f * f;
    float p = fmaf(y, 4.6630280576761255e-4f, -7.3704309457143504e-3f);   // pi^13/13!, -pi^11/11!
    p = fmaf(y, p, 8.2145886611128229e-2f);                                // pi^9/9!
    p = fmaf(y, p, -5.9926452932079208e-1f);                               // -pi^7/7!
    p = fmaf(y, p, 2.5501640398773455f);                                   // pi^5/5!
    p = fmaf(y, p, -5.1677127800499700f);                                  // -pi^3/3!
    p = fmaf(y, p, -8.7422780126189537e-8f);                               // pi - (float)pi
    sh = fmaf(f, 3.14159274101257324f, f * p);                             // (float)pi
    float c = fmaf(y, 1.9295743094039220e-3f, -2.5806891390014050e-2f);    // pi^12/12!, -pi^10/10!
    c = fmaf(y, c, 2.3533063035889312e-1f);                                // pi^8/8!
    c = fmaf(y, c, -1.3352627688545893f);                                  // -pi^6/6!
    c = fmaf(y, c, 4.0587121264167682f);                                   // pi^4/4!
    c = fmaf(y, c, -4.9348022005446793f);                                  // -pi^2/2!
    ch = fmaf(y, c, 1.0f);
}
// 2 cos(2 pi r (w + w_lo)) = 2 - 4 sin^2(pi f): relatively accurate in (2 - result) for small angles
__device__ __forceinline__ float two_cos_turns(float r, float w, float w_lo)
{
    float sh, ch;
    sincos_pi(reduce_turns(r, w, w_lo), sh, ch);
    (void)ch;
    return fmaf(-4.0f * sh, sh, 2.0f);
}
// sin(2 pi r (w + w_lo)) = 2 sin(pi f) cos(pi f)
__device__ __forceinline__ float sin_turns_accurate(float r, float w, float w_lo)
{
    float sh, ch;
    sincos_pi(reduce_turns(r, w, w_lo), sh, ch);
    return (sh + sh) * ch;
}

// accurate sin(q r)/r for one term (slow path): Taylor for |x| < 0.6 (north_star (e)), libdevice sinf otherwise
__device__ __forceinline__ float term_accurate(float qk, float r)
{
    float x = qk * r;
    if (fabsf(x) < 0.6f) {     // remainder x^12/13! < 4e-13
        float x2 = x * x;
        float p = fmaf(x2, -1.0f / 39916800.0f, 1.0f / 362880.0f);
        p = fmaf(x2, p, -1.0f / 5040.0f);
        p = fmaf(x2, p, 1.0f / 120.0f);
        p = fmaf(x2, p, -1.0f / 6.0f);
        p = fmaf(x2, p, 1.0f);
        return qk * p;
    }
    return sinf(x) / r;
}

// ---- mbarrier / bulk copy ------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(u64 *bar, int count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count)); }
__device__ __forceinline__ void mbar_expect_tx(u64 *bar, uint32_t bytes) { asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory"); }
__device__ __forceinline__ void mbar_wait(u64 *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, u64 *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// where output index k lives: q-chunk and local slot.  Recurrence chunks are residue classes mod S = 8 n_chunks
// (so every chunk can start at index 0); the direct variants use contiguous ranges.
__host__ __device__ inline void slot_of(int variant, int K, int n_chunks, int kprime, int &ch, int &l)
{
    if (variant == V_RECUR) {
        int S = 8 * n_chunks;
        ch = (kprime % S) / 8;
        l = 8 * (kprime / S) + (kprime % 8);
    } else {
        ch = kprime / K;
        l = kprime % K;
    }
}

struct ChunkConst {          // per (q-chunk) constants of the recurrence variant, rebuilt when the chunk changes
    float dq;                // theta = r * dq
    float w[8];              // general start: turns per Angstrom of the 8 MUFU start values
    float c4turn;            // general start: 4 dq / (2 pi)
    float cut2;              // r^2 below which the slow path is taken
    float qbase, qstep;      // slow path / direct: q of local slot l is computed from these (recurrence) ...
    int zs;                  // zero start usable for this chunk
    int ch;
};

template <int K, int VAR>
struct PairAcc {
    // FP32 variants: K/2 packed accumulators; F64: K doubles
    typedef typename std::conditional<VAR == V_F64, double, u64>::type elem_t;
    static constexpr int NE = (VAR == V_F64) ? K : K / 2;
    elem_t v[NE];
};

#ifndef DEBYE_FLUSH_J
#define DEBYE_FLUSH_J 4096
#endif

template <int K, int VAR>
__global__ void __launch_bounds__(DEBYE_IB, (VAR == V_F64) ? 1 : (K <= 64 ? 4 : (K <= 112 ? 3 : 2))) debye_pairs_kernel(const DevPlan *__restrict__ plan, const float4 *__restrict__ sorted, const float *__restrict__ qv,
                                                               double *__restrict__ records, int n_chunks, int is_auto, float theta_min)
{
    // ---- variant gate (decided on the device so the host never reads q) ---------------------------------------
    if (is_auto) {
        if (plan->variant_auto != VAR) return;
    } else if (VAR == V_RECUR && !plan->uniform) {
        return;   // the final kernel writes NaN in this case
    }
    constexpr bool F64 = (VAR == V_F64);
    constexpr int NW = DEBYE_IB / 32;
    __shared__ __align__(128) float4 tile[2][DEBYE_JT];
    __shared__ __align__(8) u64 mbar[2];
    __shared__ float tbuf[F64 ? 1 : NW][F64 ? 1 : 32][F64 ? 1 : 33];
    __shared__ double wsum[NW][K];
    __shared__ float qs[(VAR == V_RECUR) ? 1 : K];
    __shared__ float wtab[16];                        // recurrence, general start: start frequencies (hi[8], lo[8])    // direct variants: q of each local slot (0 for padding)

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = gridDim.x, c = blockIdx.x;
    const int N = plan->N, n_tp = plan->n_tp, Bn = plan->B, M = plan->M;
    const int64_t U1 = plan->U1;
    const int64_t Uc = U1 * n_chunks;            // units per conformer
    const int64_t U = Uc * Bn;
    if (U == 0) return;
    const int64_t u0 = debye_range_begin(U, c, G);
    const int64_t u1 = (c + 1 == G) ? U : debye_range_begin(U, c + 1, G);
    if (u0 >= u1) return;

    if (tid == 0) { mbar_init(&mbar[0], 1); mbar_init(&mbar[1], 1); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();
    uint32_t phase0 = 0, phase1 = 0;

    PairAcc<K, VAR> acc;
#pragma unroll
    for (int i = 0; i < PairAcc<K, VAR>::NE; ++i) acc.v[i] = 0;
    double run = 0.0;                 // thread k < K owns the FP64 running sum of local slot k
    int64_t curX = -1;
    int pending = 0;

    // recurrence constants
    const int uniform = plan->uniform;
    const double dq_d = plan->dq, q0_d = plan->q0;
    const int koff = plan->zero_start;           // >= 0: grid is (k + koff) dq with koff small; -1: general
    float dqf = 0.f, cut2 = 0.f, cS_unused = 0.f;
    float wS_lo = 0.f, w4_lo = 0.f, w1 = 0.f, w1_lo = 0.f;
    float wS = 0.f, w4 = 0.f;   // S dq / 2 pi and 4 dq / 2 pi (turns per Angstrom of the chain / bootstrap stride)
    float qbase_l = 0.f;      // q of local slot l (recurrence): qbase_l + (S*(l/8) + (l%8)) * dq
    int zs = 0, ch_cur = 0;
    (void)cS_unused; (void)uniform;

    auto flush = [&]() {
        // FP32 -> FP64, fixed order.  Each warp transposes 32 slots x 32 lanes through tbuf; lane l sums slot
        // 32 s + l over the 32 lanes in lane order; then threads k < K add the 4 warp sums in warp order.
        if constexpr (!F64) {
#pragma unroll
            for (int s = 0; s < (K + 31) / 32; ++s) {
#pragma unroll
                for (int t = 0; t < 32; t += 2) {
                    int l = 32 * s + t;
                    if (l < K) {
                        float lo, hi;
                        upk2(acc.v[l / 2], lo, hi);
                        tbuf[warp][t][lane] = lo;
                        tbuf[warp][t + 1][lane] = hi;
                        acc.v[l / 2] = 0;
                    }
                }
                __syncwarp();
                if (32 * s + lane < K) {
                    double sum = 0.0;
#pragma unroll
                    for (int j = 0; j < 32; ++j) sum += (double)tbuf[warp][lane][j];
                    wsum[warp][32 * s + lane] = sum;
                }
                __syncwarp();
            }
        } else {
#pragma unroll
            for (int l = 0; l < K; ++l) {
                double v = acc.v[l];
                acc.v[l] = 0;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);   // xor tree: same order every run
                if (lane == 0) wsum[warp][l] = v;
            }
        }
        __syncthreads();
        if (tid < K) {
            double s = 0.0;
#pragma unroll
            for (int w = 0; w < NW; ++w) s += wsum[w][tid];
            run += s;
        }
        __syncthreads();
    };
    auto write_record = [&](int64_t X) {
        if (tid < K) { records[((int64_t)c + X) * K + tid] = run; run = 0.0; }
    };

    int64_t u = u0;
    while (u < u1) {
        // ---- decode unit u -> (conformer, type pair, chunk, row, first j) -------------------------------------
        const int b = (int)(u / Uc);
        const int64_t w = u % Uc;
        int lo = 0, hi = n_tp;                    // largest tp with tp_prefix[tp]*n_chunks <= w
        while (hi - lo > 1) { int mid = (lo + hi) >> 1; if (plan->tp_prefix[mid] * n_chunks <= w) lo = mid; else hi = mid; }
        const int tp = lo;
        const int64_t tp_units = plan->tp_prefix[tp + 1] - plan->tp_prefix[tp];
        const int64_t w2 = w - plan->tp_prefix[tp] * n_chunks;
        const int ch = (int)(w2 / tp_units);
        const int64_t v = w2 % tp_units;
        const int ti = plan->tp_ti[tp], tj = plan->tp_tj[tp];
        const bool diag = (ti == tj);
        const int n_i = plan->n_a[ti], n_j = plan->n_a[tj];
        int row; int64_t jo, row_units;
        if (!diag) { row = (int)(v / n_j); jo = v % n_j; row_units = n_j; }
        else {
            int rl = 0, rh = debye_diag_rows(n_i);
            while (rh - rl > 1) { int mid = (rl + rh) >> 1; if (debye_diag_row_prefix(n_i, mid) <= v) rl = mid; else rh = mid; }
            row = rl; jo = v - debye_diag_row_prefix(n_i, row); row_units = (int64_t)n_i - 1 - (int64_t)row * DEBYE_IB;
        }
        const int len = (int)min((int64_t)(u1 - u), row_units - jo);
        const int64_t X = ((int64_t)b * n_tp + tp) * n_chunks + ch;

        if (X != curX) {
            if (curX >= 0) { flush(); pending = 0; write_record(curX); }
            curX = X;
            if (ch != ch_cur || u == u0) {
                ch_cur = ch;
                if constexpr (VAR == V_RECUR) {
                    const int S = 8 * n_chunks;
                    dqf = (float)dq_d;
                    zs = (koff >= 0 && n_chunks <= 2) ? 1 : 0;
                    const double qb = (koff >= 0) ? 0.0 : q0_d;          // q of k' = 0
                    qbase_l = (float)(qb + (8.0 * ch) * dq_d);
                    const int base = -S + 8 * ch;                         // k' of the first start value
                    __syncthreads();
                    if (tid < 8) {   // turns per Angstrom of the 8 general-start values, hi and lo parts
                        const double wd = (qb + (double)(base + tid) * dq_d) * 0.15915494309189535;
                        const float wh = (float)wd;
                        wtab[tid] = wh; wtab[8 + tid] = (float)(wd - (double)wh);
                    }
                    __syncthreads();
                    const double w1_d = dq_d * 0.15915494309189535;
                    w1 = (float)w1_d; w1_lo = (float)(w1_d - (double)w1);
                    const double wS_d = (double)S * dq_d * 0.15915494309189535, w4_d = 4.0 * dq_d * 0.15915494309189535;
                    wS = (float)wS_d; wS_lo = (float)(wS_d - (double)wS);
                    w4 = (float)w4_d; w4_lo = (float)(w4_d - (double)w4);
                    float rc = theta_min / fabsf(dqf);
                    cut2 = rc * rc;
                } else {
                    __syncthreads();
                    if (tid < K) { int k = ch * K + tid; qs[tid] = (k < M) ? qv[k] : 0.0f; }
                    __syncthreads();
                    float rc = theta_min / fmaxf(plan->q_small, 1e-30f);
                    cut2 = (plan->q_small > 0.f) ? rc * rc : 0.f;
                }
            }
        }

        // ---- this thread's i atom --------------------------------------------------------------------------------
        const int i_local = row * DEBYE_IB + tid;
        const bool ivalid = i_local < n_i;
        const float4 *conf = sorted + (int64_t)b * N;
        float4 pi = conf[plan->seg_off[ti] + (ivalid ? i_local : 0)];
        const int j_first = diag ? (row * DEBYE_IB + 1 + (int)jo) : (int)jo;   // index within the j type segment
        const float4 *src = conf + plan->seg_off[tj] + j_first;
        const int ntile = (len + DEBYE_JT - 1) / DEBYE_JT;

        if (tid == 0) {
            uint32_t bytes = (uint32_t)min(len, DEBYE_JT) * 16u;
            mbar_expect_tx(&mbar[0], bytes);
            bulk_g2s(&tile[0][0], src, bytes, &mbar[0]);
        }
        for (int t = 0; t < ntile; ++t) {
            const int buf = t & 1;
            if (tid == 0 && t + 1 < ntile) {
                uint32_t bytes = (uint32_t)min(len - (t + 1) * DEBYE_JT, DEBYE_JT) * 16u;
                mbar_expect_tx(&mbar[buf ^ 1], bytes);
                bulk_g2s(&tile[buf ^ 1][0], src + (t + 1) * DEBYE_JT, bytes, &mbar[buf ^ 1]);
            }
            if (buf == 0) { mbar_wait(&mbar[0], phase0); phase0 ^= 1; } else { mbar_wait(&mbar[1], phase1); phase1 ^= 1; }
            const int cnt = min(len - t * DEBYE_JT, DEBYE_JT);
            const int jl0 = j_first + t * DEBYE_JT;
            // on the diagonal, a warp whose every i is >= j has nothing to do for that j: start later
            int jj0 = 0;
            if (diag) { int first_i = row * DEBYE_IB + warp * 32; jj0 = max(0, first_i + 1 - jl0); }
            for (int jj = jj0; jj < cnt; ++jj) {
                const float4 pj = tile[buf][jj];
                const bool ok = ivalid && (!diag || (jl0 + jj > i_local));
                if constexpr (F64) {
                    double dx = (double)pj.x - (double)pi.x, dy = (double)pj.y - (double)pi.y, dz = (double)pj.z - (double)pi.z;
                    double r = sqrt(dx * dx + dy * dy + dz * dz);
                    if (ok) {
#pragma unroll
                        for (int l = 0; l < K; ++l) {
                            double qk = (double)qs[l];
                            double x = qk * r;
                            acc.v[l] += (x == 0.0) ? qk : sin(x) / r;
                        }
                    }
                } else {
                    const float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
                    const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                    const bool small = !(r2 > cut2);
                    const float r2c = fmaxf(r2, 1e-30f);
                    float rinv = rsqrt_mufu(r2c);
                    const float r = r2c * rinv;
                    rinv = (ok && !small) ? rinv : 0.0f;
                    if (__any_sync(0xffffffffu, small && ok)) {
                        if (small && ok) {
                            const float rs = sqrtf(r2);
#pragma unroll
                            for (int l = 0; l < K; ++l) {
                                float qk;
                                if constexpr (VAR == V_RECUR) qk = qbase_l + (float)(8 * n_chunks * (l / 8) + (l % 8)) * dqf;
                                else qk = qs[l];
                                float lo_, hi_;
                                upk2(acc.v[l / 2], lo_, hi_);
                                float tv = (rs == 0.0f) ? qk : term_accurate(qk, rs);
                                if (l & 1) hi_ += tv; else lo_ += tv;
                                acc.v[l / 2] = pk2(lo_, hi_);
                            }
                        }
                    }
                    if constexpr (VAR == V_RECUR) {
                        // ---- start values: u_j = sin(.)/r at the 16 indices the 4 packed chains need ---------------
                        u64 A[4], Bv[4];
                        float cS;
                        if (zs) {
                            // zero start (q_k' = k' dq, 1 or 2 residue-class chunks): v_n = sin(n theta), v_0 = 0,
                            // v_{-n} = -v_n.  sin/cos(theta/2) by polynomial, everything else by double-angle /
                            // three-term steps (each a single rounding, so relative accuracy survives small theta).
                            float sh, chh;
                            sincos_pi(reduce_turns(r, w1, w1_lo), sh, chh);
                            const float s1 = (sh + sh) * chh;                     // sin(theta)
                            const float c1 = fmaf(-4.0f * sh, sh, 2.0f);          // 2 cos(theta)
                            const float c2 = fmaf(-4.0f * s1, s1, 2.0f);          // 2 cos(2 theta)
                            const float s2 = s1 * c1;                             // sin(2 theta)
                            const float c4 = fmaf(-4.0f * s2, s2, 2.0f);          // 2 cos(4 theta)
                            // the chain coefficient 2 cos(S theta) is NOT derived from these by further doubling: the
                            // correlated roundings of that route leave a +7e-8 rad coherent phase bias after 16 steps
                            // (fp32 emulation); the direct polynomial on the reduced angle has none
                            cS = two_cos_turns(r, wS, wS_lo);
                            float u[17];
                            u[0] = 0.0f;
                            u[1] = s1 * rinv; u[2] = c1 * u[1]; u[3] = fmaf(c1, u[2], -u[1]); u[4] = c2 * u[2];
                            u[5] = fmaf(c4, u[1], u[3]); u[6] = fmaf(c4, u[2], u[2]); u[7] = fmaf(c4, u[3], u[1]); u[8] = c4 * u[4];
                            if (n_chunks == 1) {
                                // w_0 = v_0 (B), w_{-1} = -v_{-1} = +v_{8-n} (A)
                                Bv[0] = pk2(u[0], u[1]); Bv[1] = pk2(u[2], u[3]); Bv[2] = pk2(u[4], u[5]); Bv[3] = pk2(u[6], u[7]);
                                A[0] = pk2(u[8], u[7]); A[1] = pk2(u[6], u[5]); A[2] = pk2(u[4], u[3]); A[3] = pk2(u[2], u[1]);
                            } else {
                                // two chunks: stride S = 16, chunk ch owns k' = 16 m + 8 ch + (0..7)
#pragma unroll
                                for (int n = 9; n <= 16; ++n) u[n] = fmaf(c4, u[n - 4], -u[n - 8]);
                                if (ch_cur == 0) {
                                    Bv[0] = pk2(u[0], u[1]); Bv[1] = pk2(u[2], u[3]); Bv[2] = pk2(u[4], u[5]); Bv[3] = pk2(u[6], u[7]);
                                    A[0] = pk2(u[16], u[15]); A[1] = pk2(u[14], u[13]); A[2] = pk2(u[12], u[11]); A[3] = pk2(u[10], u[9]);
                                } else {
                                    Bv[0] = pk2(u[8], u[9]); Bv[1] = pk2(u[10], u[11]); Bv[2] = pk2(u[12], u[13]); Bv[3] = pk2(u[14], u[15]);
                                    A[0] = pk2(u[8], u[7]); A[1] = pk2(u[6], u[5]); A[2] = pk2(u[4], u[3]); A[3] = pk2(u[2], u[1]);
                                }
                            }
                        } else {
                            // general start (q_0 not a small multiple of dq, or more than 2 chunks): 8 accurate sines at
                            // k' = base .. base+7 (base = -S + 8 ch), then the stride-4 recurrence
                            // v_{n+4} = 2cos(4 theta) v_n - v_{n-4} walks up to k' = 8 ch .. 8 ch + 7
                            float g0[4], g1[4];
#pragma unroll
                            for (int j = 0; j < 4; ++j) {
                                g0[j] = sin_turns_accurate(r, wtab[j], wtab[8 + j]) * rinv;
                                g1[j] = sin_turns_accurate(r, wtab[4 + j], wtab[12 + j]) * rinv;
                            }
                            const float c4 = two_cos_turns(r, w4, w4_lo);                       // 2 cos(4 theta)
                            float a0[4], a1[4];
#pragma unroll
                            for (int j = 0; j < 4; ++j) { a0[j] = g0[j]; a1[j] = g1[j]; }
                            for (int st = 0; st < 2 * n_chunks; ++st) {
                                // advance one group of 4: (g0, g1) -> (g1, c4 g1 - g0)
#pragma unroll
                                for (int j = 0; j < 4; ++j) { float nx = fmaf(c4, g1[j], -g0[j]); g0[j] = g1[j]; g1[j] = nx; }
                            }
                            cS = two_cos_turns(r, wS, wS_lo);                                   // 2 cos(S theta)
                            Bv[0] = pk2(g0[0], g0[1]); Bv[1] = pk2(g0[2], g0[3]); Bv[2] = pk2(g1[0], g1[1]); Bv[3] = pk2(g1[2], g1[3]);
                            A[0] = pk2(-a0[0], -a0[1]); A[1] = pk2(-a0[2], -a0[3]); A[2] = pk2(-a1[0], -a1[1]); A[3] = pk2(-a1[2], -a1[3]);
                        }
                        const u64 cP = pk2(cS, cS), cN = pk2(-cS, -cS);
                        // ---- hot loop: w_m = sigma_m v_m with sigma = (+,+,-,-): w_{m+1} = (+/-) cS w_m + w_{m-1} --------
#pragma unroll
                        for (int m = 0; m < K / 8; ++m) {
#pragma unroll
                            for (int a = 0; a < 4; ++a) {
                                if (m & 2) acc.v[4 * m + a] = sub2(acc.v[4 * m + a], Bv[a]);
                                else acc.v[4 * m + a] = add2(acc.v[4 * m + a], Bv[a]);
                                if (m + 1 < K / 8) {
                                    u64 nx = fma2((m & 1) ? cN : cP, Bv[a], A[a]);
                                    A[a] = Bv[a];
                                    Bv[a] = nx;
                                }
                            }
                        }
                    } else if constexpr (VAR == V_MUFU) {
                        const float rt = r * 0.15915494309189535f;            // r / 2 pi: turns = q_k * rt
#pragma unroll
                        for (int l = 0; l < K; l += 2) {
                            float s0 = sin_turns_fma(rt, qs[l]) * rinv, s1 = sin_turns_fma(rt, qs[l + 1]) * rinv;
                            acc.v[l / 2] = add2(acc.v[l / 2], pk2(s0, s1));
                        }
                    } else {   // V_ACCURATE
#pragma unroll
                        for (int l = 0; l < K; l += 2) {
                            float s0 = sinf(qs[l] * r) * rinv, s1 = sinf(qs[l + 1] * r) * rinv;
                            acc.v[l / 2] = add2(acc.v[l / 2], pk2(s0, s1));
                        }
                    }
                }
            }
            __syncthreads();
        }
        pending += len;
        if (pending >= DEBYE_FLUSH_J) { flush(); pending = 0; }
        u += len;
    }
    if (curX >= 0) { flush(); write_record(curX); }
}

}  // namespace debye
