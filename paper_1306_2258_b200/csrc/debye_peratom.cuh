// debye_peratom.cuh -- the paper's general case: one form-factor row per ATOM.
//
//     I(q_m) = sum_i ff[i][m]^2 + 2 sum_{i<j} ff[i][m] ff[j][m] sin(q_m r_ij) / (q_m r_ij)          (Eq. 2)
//
// With a different f on every atom the per-type-pair factoring of the main path is gone: every term needs its own
// f_j(q_m), so the inner loop is the paper's own -- distance once per pair and q-chunk, then per q one
// sine, one multiply by 1/r and one FMA with f_j(q_m) read from shared memory -- and any q grid is allowed (no recurrence:
// it would save nothing here, the f_j load and FMA per term remain).  The bound is the XU pipe: one MUFU.SIN per term,
// 16 lanes per clock and SM.
//   thread = one i atom of a row of DEBYE_IB atoms, DEBYE_PA_KQ accumulators (one q-chunk) in registers ("private memory",
//   PAPER.md:86); j atoms stream through shared memory in tiles of DEBYE_PA_JT atoms: float4 position + DEBYE_PA_KQ form
//   factors each ("local memory", Fig. 2).  Units (one j atom against one row) are linearised q-chunk -> row ->
//   j and cut into G equal contiguous ranges, as in the main path (static, balanced, bitwise reproducible).  The FP32
//   accumulators are multiplied by f_i and reduced in FP64 in a fixed order at least every DEBYE_PA_FLUSH j atoms; a CTA
//   writes one FP64 record per q-chunk it touched and the final kernel adds the records in CTA order.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <type_traits>
#include "debye_plan.cuh"
#include "debye_pairs.cuh"

namespace debye {

#define DEBYE_PA_KQ 32           // largest q-chunk (accumulators per thread); the kernel is instantiated for 16, 20, ... 32
#define DEBYE_PA_JT 64
#ifndef DEBYE_PA_CTAS
#define DEBYE_PA_CTAS 4          // FP32 kernel: CTAs per SM
#endif
#define DEBYE_PA_FLUSH 2048
#define DEBYE_PA_SLICES 64       // self-term kernel: atom slices (grid.y)

// sum_i ff[i][m] and sum_i ff[i][m]^2 in FP64, fixed order: slice s of DEBYE_PA_SLICES takes atoms s, s + S, ... in 8
// interleaved sub-slices that are added in order.  selfbuf[s][0][m] = sum f, selfbuf[s][1][m] = sum f^2.
__global__ void __launch_bounds__(256) debye_peratom_self_kernel(const float *__restrict__ ff, int N, int M, double *__restrict__ selfbuf)
{
    pdl_wait();                            // launched with programmatic stream serialisation behind the pack kernel (debye_plan.cuh)
    pdl_trigger();
    __shared__ double p1[8][32], p2[8][32];
    const int kk = threadIdx.x & 31, sub = threadIdx.x >> 5;
    const int k = blockIdx.x * 32 + kk, s = blockIdx.y;
    double s1 = 0.0, s2 = 0.0;
    if (k < M)
        for (int64_t i = (int64_t)s * 8 + sub; i < N; i += (int64_t)DEBYE_PA_SLICES * 8) {
            const double f = (double)ff[i * M + k];
            s1 += f; s2 += f * f;
        }
    p1[sub][kk] = s1; p2[sub][kk] = s2;
    __syncthreads();
    if (sub == 0 && k < M) {
        double a = 0.0, b = 0.0;
#pragma unroll
        for (int x = 0; x < 8; ++x) { a += p1[x][kk]; b += p2[x][kk]; }
        selfbuf[((int64_t)s * 2 + 0) * M + k] = a;
        selfbuf[((int64_t)s * 2 + 1) * M + k] = b;
    }
}

// q-chunk that wastes the fewest padded slots for M q values (ties: the larger chunk, fewer distance evaluations)
__host__ __device__ inline int debye_peratom_kq(int M)
{
    int best = DEBYE_PA_KQ, best_slots = (M + DEBYE_PA_KQ - 1) / DEBYE_PA_KQ * DEBYE_PA_KQ;
    for (int kq = DEBYE_PA_KQ - 4; kq >= 16; kq -= 4) {
        const int slots = (M + kq - 1) / kq * kq;
        if (slots < best_slots) { best = kq; best_slots = slots; }
    }
    return best;
}

template <bool F64, int KQ>
__global__ void __launch_bounds__(DEBYE_IB, F64 ? 2 : DEBYE_PA_CTAS) debye_peratom_pairs_kernel(const float *__restrict__ xyz, const float *__restrict__ ff,
                                                                                      const float *__restrict__ qv, int N, int M, int n_chunks,
                                                                                      double *__restrict__ records)
{
    pdl_wait();
    typedef typename std::conditional<F64, double, float>::type acc_t;
    constexpr int JT = DEBYE_PA_JT, NW = DEBYE_IB / 32;
    __shared__ __align__(16) float4 pos[JT];
    __shared__ __align__(16) float fj[JT][KQ];
    __shared__ double wsum[NW][KQ];
    __shared__ float qmin_s[NW];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = gridDim.x, c = blockIdx.x;
    const int rows = debye_diag_rows(N);
    const int64_t U1 = rows > 0 ? debye_diag_row_prefix(N, rows) : 0;
    const int64_t U = U1 * n_chunks;
    if (U == 0) return;
    const int64_t u0 = debye_range_begin(U, c, G);
    const int64_t u1 = (c + 1 == G) ? U : debye_range_begin(U, c + 1, G);
    if (u0 >= u1) return;

    // smallest non-zero |q|: pairs with q_small * r <= 0.004 take the accurate path (MUFU.SIN loses relative accuracy there)
    float cut2 = 0.f;
    if constexpr (!F64) {
        float qsm = 3.0e38f;
        for (int k = tid; k < M; k += DEBYE_IB) { const float a = fabsf(qv[k]); if (a > 0.f) qsm = fminf(qsm, a); }
        for (int o = 16; o > 0; o >>= 1) qsm = fminf(qsm, __shfl_xor_sync(0xffffffffu, qsm, o));
        if (lane == 0) qmin_s[warp] = qsm;
        __syncthreads();
        qsm = fminf(fminf(qmin_s[0], qmin_s[1]), fminf(qmin_s[2], qmin_s[3]));
        if (qsm < 3.0e38f) { const float rcut = 0.004f / qsm; cut2 = rcut * rcut; }
    }

    acc_t acc[KQ];
    float qr[KQ];
#pragma unroll
    for (int l = 0; l < KQ; ++l) { acc[l] = 0; qr[l] = 0.f; }
    double run = 0.0;                  // thread l < KQ: FP64 running sum of q slot l of the current chunk
    int ch_cur = -1;

    int64_t u = u0;
    while (u < u1) {
        // ---- decode unit u -> (q-chunk, row, first j) ------------------------------------------------------------------
        const int ch = (int)(u / U1);
        const int64_t v = u - (int64_t)ch * U1;
        int rl = 0, rh = rows;
        while (rh - rl > 1) { const int mid = (rl + rh) >> 1; if (debye_diag_row_prefix(N, mid) <= v) rl = mid; else rh = mid; }
        const int row = rl;
        const int64_t jo = v - debye_diag_row_prefix(N, row);
        const int64_t row_units = (int64_t)N - 1 - (int64_t)row * DEBYE_IB;
        const int len = (int)min(min((int64_t)(u1 - u), row_units - jo), (int64_t)DEBYE_PA_FLUSH);
        const int k0 = ch * KQ;
        if (ch != ch_cur) {
            if (ch_cur >= 0 && tid < KQ) { records[((int64_t)c + ch_cur) * KQ + tid] = run; run = 0.0; }
            ch_cur = ch;
#pragma unroll
            for (int l = 0; l < KQ; ++l) qr[l] = (k0 + l < M) ? qv[k0 + l] : 0.f;
        }
        const int i = row * DEBYE_IB + tid;
        const bool ivalid = i < N;
        const float *xi = xyz + 3 * (int64_t)(ivalid ? i : 0);
        const float pix = xi[0], piy = xi[1], piz = xi[2];
        const int j_first = row * DEBYE_IB + 1 + (int)jo;

        for (int t0 = 0; t0 < len; t0 += JT) {
            const int cnt = min(len - t0, JT), jg0 = j_first + t0;
            __syncthreads();                                   // the previous tile has been consumed
            if (tid < cnt) { const float *s = xyz + 3 * (int64_t)(jg0 + tid); pos[tid] = make_float4(s[0], s[1], s[2], 0.f); }
#pragma unroll 4
            for (int e = tid; e < JT * KQ; e += DEBYE_IB) {
                const int jj = e / KQ, l = e % KQ;
                fj[jj][l] = (jj < cnt && k0 + l < M) ? ff[(int64_t)(jg0 + jj) * M + k0 + l] : 0.f;
            }
            __syncthreads();
            // rows are diagonal blocks of the j > i triangle: a warp whose every i is >= j has nothing to do for that j
            const int jj0 = max(0, row * DEBYE_IB + warp * 32 + 1 - jg0);
            if constexpr (!F64) {
                // Software pipeline as mufu_tile (debye_pairs.cuh): the geometry of pair jj + 1 (tile load, distance, MUFU.RSQ) sits
                // in the basic block of the KQ terms of pair jj, so a MUFU.SIN is always ready to issue; pairs below the accuracy
                // cut contribute zero here (1/r := 0) and are redone term by term in a rescan of the tile that runs only if
                // some lane met one (a vote and a branch per pair would end the block at every pair).
                if (jj0 < cnt) {
                    bool had_slow = false;
                    auto geom = [&](const int jj, float &rt, float &rinv) {
                        const float4 pj = pos[min(jj, cnt - 1)];
                        const float dx = pj.x - pix, dy = pj.y - piy, dz = pj.z - piz;
                        const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                        const bool small = !(r2 > cut2), ok = ivalid && (jg0 + jj > i) && jj < cnt;
                        const float r2c = fmaxf(r2, 1e-30f);
                        const float ri = rsqrt_mufu(r2c);
                        rt = (r2c * ri) * 0.15915494309189535f;                       // r / 2 pi: turns = q_k * rt
                        rinv = (ok && !small) ? ri : 0.0f;
                        had_slow = had_slow || (small && ok);
                    };
                    float rt, rinv;
                    geom(jj0, rt, rinv);
                    for (int jj = jj0; jj < cnt; ++jj) {
                        float rtn, rinvn;
                        geom(jj + 1, rtn, rinvn);
#pragma unroll
                        for (int l = 0; l < KQ; l += 4) {
                            const float4 f4 = *reinterpret_cast<const float4 *>(&fj[jj][l]);
                            acc[l + 0] = fmaf(sin_turns_fma(rt, qr[l + 0]) * rinv, f4.x, acc[l + 0]);
                            acc[l + 1] = fmaf(sin_turns_fma(rt, qr[l + 1]) * rinv, f4.y, acc[l + 1]);
                            acc[l + 2] = fmaf(sin_turns_fma(rt, qr[l + 2]) * rinv, f4.z, acc[l + 2]);
                            acc[l + 3] = fmaf(sin_turns_fma(rt, qr[l + 3]) * rinv, f4.w, acc[l + 3]);
                        }
                        rt = rtn; rinv = rinvn;
                    }
                    if (__any_sync(0xffffffffu, had_slow)) {
                        if (had_slow) {
                            for (int jj = jj0; jj < cnt; ++jj) {
                                const float4 pj = pos[jj];
                                const float dx = pj.x - pix, dy = pj.y - piy, dz = pj.z - piz;
                                const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                                if (ivalid && (jg0 + jj > i) && !(r2 > cut2)) {
                                    const float rs = sqrtf(r2);
#pragma unroll
                                    for (int l = 0; l < KQ; ++l) {
                                        const float qk = qr[l];
                                        const float tv = (rs == 0.0f) ? qk : term_accurate(qk, rs);
                                        acc[l] = fmaf(fj[jj][l], tv, acc[l]);
                                    }
                                }
                            }
                        }
                    }
                }
            } else
            for (int jj = jj0; jj < cnt; ++jj) {
                const float4 pj = pos[jj];
                const bool ok = ivalid && (jg0 + jj > i);
                if constexpr (F64) {
                    const double dx = (double)pj.x - (double)pix, dy = (double)pj.y - (double)piy, dz = (double)pj.z - (double)piz;
                    const double r = sqrt(dx * dx + dy * dy + dz * dz);
                    if (ok) {
#pragma unroll
                        for (int l = 0; l < KQ; ++l) {
                            const double qk = (double)qr[l], x = qk * r;
                            const double tv = (x == 0.0) ? qk : sin(x) / r;          // sin(q r)/r -> q as r -> 0
                            acc[l] += (double)fj[jj][l] * tv;
                        }
                    }
                }
            }
        }
        // ---- flush: times f_i, FP64, fixed order (xor tree over the lanes, then the warps in order) ---------------------------
        {
            const float *fi = ff + (int64_t)(ivalid ? i : 0) * M + k0;
#pragma unroll
            for (int l = 0; l < KQ; ++l) {
                double vv = (ivalid && k0 + l < M) ? (double)acc[l] * (double)fi[l] : 0.0;
                acc[l] = 0;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) vv += __shfl_xor_sync(0xffffffffu, vv, o);
                if (lane == 0) wsum[warp][l] = vv;
            }
            __syncthreads();
            if (tid < KQ) {
                double s = 0.0;
#pragma unroll
                for (int w = 0; w < NW; ++w) s += wsum[w][tid];
                run += s;
            }
        }
        u += len;
    }
    if (ch_cur >= 0 && tid < KQ) records[((int64_t)c + ch_cur) * KQ + tid] = run;
}

// I[m] = sum_i f^2 + (2 / q_m) sum over CTAs of their records   (q_m != 0);   I[m] = (sum_i f)^2   (q_m == 0)
// Block = 32 q indices x DEBYE_PA_FS slices: thread (kk, sl) adds the sl-th of DEBYE_PA_FS equal parts of the CTA range
// that touched q index k (8 record loads in flight, added in CTA order); the parts are then added in slice order, so the
// order is a fixed function of (N, M, G) and the result is bitwise reproducible.
#define DEBYE_PA_FS 8
// Batches (debye_profile_peratom_batch): blockIdx.y is the conformer; the unit line is conformer -> chunk -> row -> j.
// rplan != nullptr: the records come from debye_peratom_recur_kernel (debye_peratom_recur.cuh): chain slots (slot_of) holding
// sums of 2 sin(q r)/r; a wrong grid hint (rplan->bad) gives NaN.
struct PeratomPlan;
__global__ void __launch_bounds__(32 * DEBYE_PA_FS) debye_peratom_final_kernel(const double *__restrict__ records, const double *__restrict__ selfbuf,
                                                                                 const float *__restrict__ qv, int N, int M, int n_chunks, int G, int KQ,
                                                                                 double *__restrict__ out, const int32_t *__restrict__ rplan)
{
    __shared__ double part[DEBYE_PA_FS][32];
    pdl_wait();
    const int kk = threadIdx.x & 31, sl = threadIdx.x >> 5;
    const int k = blockIdx.x * 32 + kk;
    const int b = blockIdx.y, Bn = gridDim.y;
    out += (int64_t)b * M;
    const int rows = debye_diag_rows(N);
    const int64_t U1 = rows > 0 ? debye_diag_row_prefix(N, rows) : 0;
    const bool recur = rplan != nullptr;
    const bool bad = recur && rplan[0] != 0;                 // PeratomPlan::bad, ::koff are its first two int32
    double s = 0.0;
    if (k < M && U1 > 0 && qv[k] != 0.0f && !bad) {
        int ch = k / KQ, l = k % KQ;
        if (recur) slot_of(V_RECUR, KQ, n_chunks, k + rplan[1] - 1, ch, l);
        const int64_t X = (int64_t)b * n_chunks + ch;          // record slot of (conformer, chunk)
        const int64_t U = U1 * n_chunks * Bn, ub = X * U1, ue = ub + U1 - 1;
        const DebyeRanges ranges(U, G);
        if (U >= G) {           // every CTA owns at least one unit: all CTAs between the owners took part
            const int c_lo = ranges.owner(ub), c_hi = ranges.owner(ue);
            const int n = c_hi - c_lo + 1, per = (n + DEBYE_PA_FS - 1) / DEBYE_PA_FS;
            const int cb = c_lo + sl * per, ce = min(c_hi + 1, cb + per);
            const double *rp = records + ((int64_t)cb + X) * KQ + l;
            int c = cb;
            for (; c + 8 <= ce; c += 8, rp += 8 * (int64_t)KQ) {
                double r[8];
#pragma unroll
                for (int x = 0; x < 8; ++x) r[x] = rp[x * (int64_t)KQ];
#pragma unroll
                for (int x = 0; x < 8; ++x) s += r[x];
            }
            for (; c < ce; ++c, rp += KQ) s += rp[0];
        } else if (sl == 0) {   // fewer units than CTAs: each unit has its own CTA
            for (int64_t u = ub; u <= ue; ++u) s += records[((int64_t)ranges.owner(u) + X) * KQ + l];
        }
    }
    part[sl][kk] = s;
    __syncthreads();
    if (sl != 0 || k >= M) return;
    double s1 = 0.0, s2 = 0.0, tot = 0.0;
    for (int x = 0; x < DEBYE_PA_SLICES; ++x) { s1 += selfbuf[((int64_t)x * 2 + 0) * M + k]; s2 += selfbuf[((int64_t)x * 2 + 1) * M + k]; }
#pragma unroll
    for (int x = 0; x < DEBYE_PA_FS; ++x) tot += part[x][kk];
    const double qk = (double)qv[k];
    if (bad) { out[k] = __longlong_as_double(0x7ff8000000000000LL); return; }
    out[k] = (qk == 0.0) ? s1 * s1 : s2 + (recur ? 1.0 : 2.0) * tot / qk;
}

}  // namespace debye
