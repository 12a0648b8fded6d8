// debye_aux.cuh -- setup (S0/S1), pack (S0) and final+epilogue (S7) kernels of libdebye.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cmath>
#include "debye_plan.cuh"
#include "debye_pairs.cuh"

namespace debye {

#define DEBYE_SETUP_THREADS 1024

// S0 + S1.  One CTA: type histogram, segment offsets, stable counting-sort permutation, q-grid analysis and the
// unit prefix per type pair.  Stable = atoms of one type keep their input order, so the sorted layout (and with
// it every rounding in the pair sums) is a pure function of the input.
// perm[p] = original index of the atom at sorted position p.
__global__ void __launch_bounds__(DEBYE_SETUP_THREADS) debye_setup_kernel(DevPlan *plan, const int32_t *__restrict__ type, const float *__restrict__ q,
                                                                            int32_t *__restrict__ perm, int N, int T, int M, int B, int rec_capacity /* K * n_chunks of the recurrence */)
{
    __shared__ int cnt[DEBYE_MAX_TYPES_I];
    __shared__ int base[DEBYE_MAX_TYPES_I + 1];
    __shared__ int wcnt[DEBYE_SETUP_THREADS / 32][DEBYE_MAX_TYPES_I];
    __shared__ float red[DEBYE_SETUP_THREADS / 32];
    __shared__ float red2[DEBYE_SETUP_THREADS / 32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid < DEBYE_MAX_TYPES_I) cnt[tid] = 0;
    __syncthreads();
    for (int i = tid; i < N; i += blockDim.x) atomicAdd(&cnt[type[i]], 1);
    __syncthreads();
    if (tid == 0) {
        int s = 0;
        for (int t = 0; t < T; ++t) { base[t] = s; plan->seg_off[t] = s; plan->n_a[t] = cnt[t]; s += cnt[t]; }
        base[T] = s;
        for (int t = T; t <= DEBYE_MAX_TYPES_I; ++t) plan->seg_off[t] = s;
        for (int t = T; t < DEBYE_MAX_TYPES_I; ++t) plan->n_a[t] = 0;
        plan->N = N; plan->T = T; plan->M = M; plan->B = B; plan->n_tp = T * (T + 1) / 2;
        // units per type pair; the side with less padding waste becomes the row (i) side
        int64_t pre = 0;
        int tp = 0;
        for (int a = 0; a < T; ++a)
            for (int b2 = a; b2 < T; ++b2, ++tp) {
                int na = cnt[a], nb = cnt[b2];
                int64_t units;
                int ti = a, tj = b2;
                if (a == b2) {
                    int rows = debye_diag_rows(na);
                    units = rows > 0 ? debye_diag_row_prefix(na, rows) : 0;
                } else {
                    int64_t ra = (na + DEBYE_IB - 1) / DEBYE_IB, rb = (nb + DEBYE_IB - 1) / DEBYE_IB;
                    int64_t ua = ra * nb, ub = rb * na;          // rows x j atoms
                    if (ub < ua) { ti = b2; tj = a; units = ub; } else units = ua;
                    if (na == 0 || nb == 0) units = 0;
                }
                plan->tp_ti[tp] = ti; plan->tp_tj[tp] = tj; plan->tp_prefix[tp] = pre;
                pre += units;
            }
        plan->tp_prefix[tp] = pre;
        for (int x = tp + 1; x <= DEBYE_MAX_TP; ++x) plan->tp_prefix[x] = pre;
        plan->U1 = pre;
    }
    __syncthreads();
    // ---- stable counting sort, 1024 atoms per step --------------------------------------------------------------
    for (int start = 0; start < N; start += blockDim.x) {
        const int i = start + tid;
        const int t = (i < N) ? type[i] : -1;
        for (int x = lane; x < T; x += 32) wcnt[warp][x] = 0;
        __syncwarp();
        unsigned peers = __match_any_sync(0xffffffffu, t);
        int rank_in_warp = __popc(peers & ((1u << lane) - 1));
        if (t >= 0 && rank_in_warp == 0) wcnt[warp][t] = __popc(peers);
        __syncthreads();
        int before = 0;
        if (t >= 0) {
            for (int w = 0; w < warp; ++w) before += wcnt[w][t];
            perm[base[t] + before + rank_in_warp] = i;
        }
        __syncthreads();
        if (tid < T) { int s = 0; for (int w = 0; w < DEBYE_SETUP_THREADS / 32; ++w) s += wcnt[w][tid]; base[tid] += s; }
        __syncthreads();
    }
    // ---- q grid analysis -------------------------------------------------------------------------------------------
    const double q0 = (double)q[0];
    double dq = (M > 1) ? ((double)q[M - 1] - q0) / (double)(M - 1) : (q0 != 0.0 ? q0 : 1.0);
    float dev = 0.f, qsm = 3.0e38f, qmax = 0.f;
    for (int k = tid; k < M; k += blockDim.x) {
        double qk = (double)q[k];
        dev = fmaxf(dev, (float)fabs(qk - (q0 + k * dq)));
        float aq = fabsf((float)qk);
        if (aq > 0.f) qsm = fminf(qsm, aq);
        qmax = fmaxf(qmax, aq);
    }
    for (int o = 16; o > 0; o >>= 1) { dev = fmaxf(dev, __shfl_xor_sync(0xffffffffu, dev, o)); qsm = fminf(qsm, __shfl_xor_sync(0xffffffffu, qsm, o)); qmax = fmaxf(qmax, __shfl_xor_sync(0xffffffffu, qmax, o)); }
    if (lane == 0) { red[warp] = dev; red2[warp] = qsm; }
    __syncthreads();
    __shared__ float qmax_s[DEBYE_SETUP_THREADS / 32];
    if (lane == 0) qmax_s[warp] = qmax;
    __syncthreads();
    if (tid == 0) {
        float d = 0.f, s = 3.0e38f, mx = 0.f;
        for (int w = 0; w < DEBYE_SETUP_THREADS / 32; ++w) { d = fmaxf(d, red[w]); s = fminf(s, red2[w]); mx = fmaxf(mx, qmax_s[w]); }
        // uniform if every q[k] is within 2 float ulps (of the largest |q|) of the line through the end points
        int uni = (dq != 0.0) && (d <= 2.4e-7f * fmaxf(mx, 1e-30f));
        int koff = -1;
        if (uni) {
            double ko = q0 / dq;
            double kr = rint(ko);
            if (kr >= 0.0 && kr <= 8.0 && fabs(ko - kr) <= 1e-6 * fmax(1.0, kr) && (int)kr + M <= rec_capacity) koff = (int)kr;
        }
        plan->uniform = uni;
        plan->zero_start = koff;
        plan->q0 = q0;
        plan->dq = dq;
        plan->q_small = (s < 3.0e38f) ? s : 0.f;
        plan->variant_auto = uni ? V_RECUR : V_MUFU;
    }
}

// S0: gather coordinates into type-sorted float4 (x, y, z, bits(type)), all conformers.
__global__ void debye_pack_kernel(const DevPlan *__restrict__ plan, const float *__restrict__ xyz, const int32_t *__restrict__ type, const int32_t *__restrict__ perm,
                                  float4 *__restrict__ sorted, int N, int B)
{
    const int64_t total = (int64_t)N * B;
    for (int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; g < total; g += (int64_t)gridDim.x * blockDim.x) {
        const int b = (int)(g / N), p = (int)(g % N);
        const int i = perm[p];
        const float *s = xyz + ((int64_t)b * N + i) * 3;
        sorted[g] = make_float4(s[0], s[1], s[2], __int_as_float(type[i]));
    }
}

// number of unordered pairs of type pair (a, b)
__device__ __forceinline__ double pair_count(int na, int nb, bool diag) { return diag ? 0.5 * (double)na * (double)(na - 1) : (double)na * (double)nb; }

// S7: fixed-order FP64 sum of the per-CTA records, then the form-factor epilogue
//   I(q_k) = sum_a n_a F_a^2 + 2 sum_{a<=b} F_a F_b S_ab(q_k),   S_ab = (1/q_k) sum sin(q_k r)/r  (q_k != 0), #pairs (q_k == 0).
// Block = (conformer, tile of 32 q indices); thread (kk, g) handles q index k0 + kk and the type pairs g, g+8, ... in
// increasing order; the 8 partial sums are then added in g order.  Every order is fixed, so the result is bitwise
// reproducible.  Record reads are coalesced over kk.  mode 0: write I_out[b][k]; mode 1: write S_out[b][tp][k].
#define DEBYE_FINAL_G 8
__global__ void __launch_bounds__(32 * DEBYE_FINAL_G) debye_final_kernel(const DevPlan *__restrict__ plan, const double *__restrict__ records,
                                                                            const float *__restrict__ fftab, const float *__restrict__ q, double *__restrict__ out,
                                                                            int is_auto, int variant0, int K0, int nc0, int G0, int variant1, int K1, int nc1, int G1,
                                                                            int mode)
{
    __shared__ double part[DEBYE_FINAL_G][32];
    const int M = plan->M, Bn = plan->B, T = plan->T, n_tp = plan->n_tp;
    const int ktiles = (M + 31) / 32;
    const int b = blockIdx.x / ktiles, k = (blockIdx.x % ktiles) * 32 + (threadIdx.x & 31), g = threadIdx.x >> 5;
    const bool live = k < M;
    // automatic mode: two pairs kernels were launched and the device ran the one named by plan->variant_auto
    const bool second = is_auto && plan->variant_auto == variant1;
    const int variant = second ? variant1 : variant0, K = second ? K1 : K0, n_chunks = second ? nc1 : nc0, G = second ? G1 : G0;
    const bool bad = (variant == V_RECUR && !plan->uniform);          // forced recurrence on a non-uniform grid -> NaN
    const double nan = __longlong_as_double(0x7ff8000000000000LL);
    double I = 0.0;
    if (live) {
        int kprime = k;
        if (variant == V_RECUR && plan->zero_start > 0) kprime = k + plan->zero_start;
        int ch, l;
        slot_of(variant, K, n_chunks, kprime, ch, l);
        const double qk = (double)q[k];
        const int64_t U1 = plan->U1, Uc = U1 * n_chunks, U = Uc * Bn;
        // type pair index -> (a, b2): walk rows of the upper triangle
        int a = 0, rowstart = 0;
        for (int tp = g; tp < n_tp; tp += DEBYE_FINAL_G) {
            while (tp >= rowstart + (T - a)) { rowstart += T - a; ++a; }
            const int b2 = a + (tp - rowstart);
            double S;
            const int64_t units = plan->tp_prefix[tp + 1] - plan->tp_prefix[tp];
            if (bad) S = nan;
            else if (qk == 0.0 || units == 0) S = pair_count(plan->n_a[a], plan->n_a[b2], a == b2);
            else {
                const int64_t ub = (int64_t)b * Uc + plan->tp_prefix[tp] * n_chunks + (int64_t)ch * units;
                const int64_t ue = ub + units - 1;
                const int64_t X = ((int64_t)b * n_tp + tp) * n_chunks + ch;
                double s = 0.0;
                if (U >= G) {           // every CTA owns at least one unit: all CTAs between the owners took part
                    const int c_lo = debye_owner(U, G, ub), c_hi = debye_owner(U, G, ue);
#pragma unroll 4
                    for (int c = c_lo; c <= c_hi; ++c) s += records[((int64_t)c + X) * K + l];
                } else {                // fewer units than CTAs: each unit has its own CTA
                    for (int64_t u = ub; u <= ue; ++u) s += records[((int64_t)debye_owner(U, G, u) + X) * K + l];
                }
                S = (variant == V_RECUR ? 0.5 * s : s) / qk;     // the recurrence kernel accumulates 2 sin(q r)/r
            }
            if (mode == 0) I += 2.0 * (double)fftab[a * M + k] * (double)fftab[b2 * M + k] * S;
            else out[((int64_t)b * n_tp + tp) * M + k] = S;
        }
    }
    if (mode != 0) return;
    part[g][threadIdx.x & 31] = I;
    __syncthreads();
    if (g == 0 && live) {
        double tot = 0.0;
        for (int a = 0; a < T; ++a) { const double fa = (double)fftab[a * M + k]; tot += (double)plan->n_a[a] * fa * fa; }
#pragma unroll
        for (int gg = 0; gg < DEBYE_FINAL_G; ++gg) tot += part[gg][threadIdx.x & 31];
        out[(int64_t)b * M + k] = tot;
    }
}

}  // namespace debye
