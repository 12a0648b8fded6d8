// debye_peratom_small.cuh -- per-ATOM form factors, ONE launch for one small structure (N <= 2048 atoms, at most 128 chain indices).
//
// PAPER.md:44, 82 (one form-factor row per atom: the paper's general case), :25 (a refinement calls the profile 10^5+ times),
// :104 (for small proteins the overheads dominate).  debye_profile_peratom on a 1000-atom structure is four launches (re-lay the
// table, self terms, pairs, final): 42 us, of which ~5 us are arithmetic.  Here, for a hinted grid q_k = (k + koff) dq with one
// chunk of chain indices, every CTA
//   1. loads all positions into shared memory (no sort: there are no types) and checks the grid hint;
//   2. runs its share of the unit line (row of 128 i atoms x j atom, the j > i triangle) through the chain recurrence of
//      debye_peratom_recur.cuh (peratom_tile): the j atoms' form-factor rows are staged per tile straight from ff[N][M] -- with one
//      chunk the chain slot of q_k is k + koff - 1, a contiguous stretch of the row -- with the chains' sign pattern applied;
//      at the end of every row segment the accumulators are multiplied by f_i and reduced in FP64 in a fixed order;
//   3. writes one FP64 record and waits at a grid-wide barrier (cooperative launch, at most one CTA per SM);
//   4. CTA k then computes output q_k: the self terms sum_i f^2 (or (sum_i f)^2 for q = 0) and the records of its slot in CTA
//      order, both by fixed-order trees.
// Fixed unit ranges and fixed orders: bitwise reproducible.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cooperative_groups.h>
#include "debye_plan.cuh"
#include "debye_pairs.cuh"
#include "debye_peratom_recur.cuh"

namespace debye {

#define DEBYE_PAS_NMAX 2048
#define DEBYE_PAS_JT 32           // j atoms per staged tile of form-factor rows
#define DEBYE_PAS_GMAX 256

__host__ __device__ inline size_t debye_peratom_small_dyn_smem(int N, int K)
{
    return (size_t)((N + 7) / 8 * 8 + 8) * 16 + (size_t)DEBYE_PAS_JT * K * 4;
}

// fixed-order sum of one double per thread over the CTA (pairwise tree over thread index): every thread gets the total
__device__ __forceinline__ double pas_block_sum(double v, double *red /* [DEBYE_IB] shared */, const int tid)
{
    __syncthreads();
    red[tid] = v;
    __syncthreads();
#pragma unroll
    for (int o = DEBYE_IB / 2; o > 0; o >>= 1) {
        if (tid < o) red[tid] += red[tid + o];
        __syncthreads();
    }
    return red[0];
}

template <int K>
__global__ void __launch_bounds__(DEBYE_IB, K <= DEBYE_PAR_K3 ? 3 : 2) debye_peratom_small_kernel(const float *__restrict__ xyz, const float *__restrict__ ff, const float *__restrict__ q,
                                                                                                   const int N, const int M, const int hint_class,
                                                                                                   double *__restrict__ records, double *__restrict__ out)
{
    constexpr int NW = DEBYE_IB / 32, JT = DEBYE_PAS_JT;
    extern __shared__ __align__(16) unsigned char dyn[];
    const int npad = (N + 7) / 8 * 8 + 8;
    float4 *pos = reinterpret_cast<float4 *>(dyn);
    float *tf = reinterpret_cast<float *>(dyn + (size_t)npad * 16);          // [JT][K], pre-signed rows of the tile's j atoms
    __shared__ double wsum[NW][K];
    __shared__ float tbuf[NW][32][33];
    __shared__ double red[DEBYE_IB];
    __shared__ int s_dev, s_qmax, s_bad, s_koff;
    __shared__ double s_dq;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = gridDim.x, c = blockIdx.x;

    // ---- 1. positions into shared memory; the q grid must be the one the hint promised ----------------------------------------
    if (tid == 0) { s_dev = 0; s_qmax = 0; }
    for (int i = tid; i < npad; i += DEBYE_IB) {
        float4 p = make_float4(0.f, 0.f, 0.f, 0.f);
        if (i < N) { const float *s = xyz + (size_t)i * 3; p = make_float4(s[0], s[1], s[2], 0.f); }
        pos[i] = p;
    }
    const double q0 = (double)q[0];
    const double dq = debye_grid_dq(q0, (double)q[M - 1], M);
    {
        float dev = 0.f, qmax = 0.f;
        for (int k = tid; k < M; k += DEBYE_IB) {
            const double qk = (double)q[k];
            dev = fmaxf(dev, debye_grid_dev(qk, k, q0, dq));
            qmax = fmaxf(qmax, fabsf((float)qk));
        }
        for (int o = 16; o > 0; o >>= 1) { dev = fmaxf(dev, __shfl_xor_sync(0xffffffffu, dev, o)); qmax = fmaxf(qmax, __shfl_xor_sync(0xffffffffu, qmax, o)); }
        __syncthreads();
        if (lane == 0) { atomicMax(&s_dev, __float_as_int(dev)); atomicMax(&s_qmax, __float_as_int(qmax)); }   // non-negative floats order like ints
    }
    __syncthreads();
    if (tid == 0) {
        const int cls = debye_grid_class(q0, dq, __int_as_float(s_dev), __int_as_float(s_qmax));
        s_koff = cls; s_dq = dq;
        s_bad = (cls != hint_class || cls < 0) ? 1 : 0;      // the host sized K for the promised grid
    }
    __syncthreads();
    const bool bad = s_bad != 0;
    const int koff = s_koff;

    // ---- 2. this CTA's share of the unit line ------------------------------------------------------------------------------------
    const int rows = debye_diag_rows(N);
    const int U = (bad || rows == 0) ? 0 : (int)debye_diag_row_prefix(N, rows);
    RecurConst rc;
    {
        const double w1_d = s_dq * 0.15915494309189535;
        rc.w1 = (float)w1_d; rc.w1_lo = (float)(w1_d - (double)rc.w1);
        rc.wS = rc.wS_lo = rc.w4 = rc.w4_lo = 0.f;
        rc.smult = 8.0f; rc.n_chunks = 1;
        const float rcut = 0.002f / fabsf((float)s_dq);
        rc.cut2 = rcut * rcut;
    }
    u64 acc[K / 2];
#pragma unroll
    for (int i = 0; i < K / 2; ++i) acc[i] = 0;
    double run = 0.0;                  // thread l < K: FP64 running sum of chain slot l
    if (U > 0) {
        int u = (int)debye_range_begin(U, c, G);
        const int u1 = (c + 1 == G) ? U : (int)debye_range_begin(U, c + 1, G);
        while (u < u1) {
            int rl = 0, rh = rows;
            while (rh - rl > 1) { const int mid = (rl + rh) >> 1; if ((int)debye_diag_row_prefix(N, mid) <= u) rl = mid; else rh = mid; }
            const int row = rl;
            const int jo = u - (int)debye_diag_row_prefix(N, row);
            const int row_units = N - 1 - row * DEBYE_IB;
            const int len = min(min(u1 - u, row_units - jo), DEBYE_PAR_FLUSH);
            const int i = row * DEBYE_IB + tid;
            const bool ivalid = i < N;
            const float4 pi = pos[ivalid ? i : 0];
            const int j_first = row * DEBYE_IB + 1 + jo;
            for (int t0 = 0; t0 < len; t0 += JT) {
                const int cnt = min(len - t0, JT), jl0 = j_first + t0;
                __syncthreads();                                   // the previous tile's rows have been consumed
                for (int e = tid; e < JT * K; e += DEBYE_IB) {     // row jj of the tile: slot l holds sigma_m ff[j][l + 1 - koff]
                    const int jj = e / K, l = e - jj * K;
                    const int k = l + 1 - koff;
                    float v = (jj < cnt && k >= 0 && k < M) ? ff[(size_t)(jl0 + jj) * M + k] : 0.f;
                    tf[e] = ((l >> 3) & 2) ? -v : v;
                }
                __syncthreads();
                const int jj0 = max(0, row * DEBYE_IB + warp * 32 + 1 - jl0);
                if (jj0 < cnt && row * DEBYE_IB + warp * 32 < N) {
                    const int jmin = ivalid ? max(0, i + 1 - jl0) : 0x7fffffff;
                    const bool had_slow = peratom_tile<K, PM_C1>(acc, pos + jl0, tf, jj0, cnt, pi, jmin, rc);
                    // pairs below the small-theta cut and coincident atoms contributed zero above: term by term (rare)
                    if (__any_sync(0xffffffffu, had_slow)) {
                        if (had_slow) {
                            for (int j = max(jj0, jmin); j < cnt; ++j) {
                                const float4 pj = pos[jl0 + j];
                                const float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
                                const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                                if (!(fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, 1e-30f))) > rc.cut2)) {
                                    const float rs = sqrtf(r2);
#pragma unroll
                                    for (int l = 0; l < K; ++l) {
                                        const float qk = (float)((double)(l + 1) * s_dq);
                                        float tv = 2.0f * ((rs == 0.0f) ? qk : term_accurate(qk, rs));     // the chains accumulate 2 sin(q r)/r
                                        if ((l >> 3) & 2) tv = -tv;                                         // the staged row carries sigma_m
                                        float lo, hi;
                                        upk2(acc[l / 2], lo, hi);
                                        if (l & 1) hi = fmaf(tf[j * K + l], tv, hi); else lo = fmaf(tf[j * K + l], tv, lo);
                                        acc[l / 2] = pk2(lo, hi);
                                    }
                                }
                            }
                        }
                    }
                }
            }
            // ---- flush: times f_i (sigma^2 = 1: the raw row), then FP64 in a fixed order: per warp the products are transposed
            // through shared memory, lane l adds slot 32 s + l over the 32 i atoms (four interleaved partial sums), then the warps in
            // order.  (An xor-shuffle tree over the lanes in FP64, as in the large kernel, took 4 us per flush here: 10 64-bit
            // shuffles per slot pair; the kernel flushes once per row segment, and the slowest CTA holds the grid barrier.)
            {
                const float *fi = ff + (size_t)(ivalid ? i : 0) * M;
#pragma unroll
                for (int s = 0; s < (K + 31) / 32; ++s) {
#pragma unroll
                    for (int t = 0; t < 32; t += 2) {
                        const int l = 32 * s + t;
                        if (l < K) {
                            float lo, hi;
                            upk2(acc[l / 2], lo, hi);
                            acc[l / 2] = 0;
                            const int k0 = l + 1 - koff, k1 = l + 2 - koff;
                            const float f0 = (ivalid && k0 >= 0 && k0 < M) ? fi[k0] : 0.f, f1 = (ivalid && k1 >= 0 && k1 < M) ? fi[k1] : 0.f;
                            tbuf[warp][t][lane] = lo * f0;
                            tbuf[warp][t + 1][lane] = hi * f1;
                        }
                    }
                    __syncwarp();
                    if (32 * s + lane < K) {
                        double p0 = 0.0, p1 = 0.0, p2 = 0.0, p3 = 0.0;
#pragma unroll
                        for (int x = 0; x < 32; x += 4) {
                            p0 += (double)tbuf[warp][lane][x]; p1 += (double)tbuf[warp][lane][x + 1];
                            p2 += (double)tbuf[warp][lane][x + 2]; p3 += (double)tbuf[warp][lane][x + 3];
                        }
                        wsum[warp][32 * s + lane] = (p0 + p1) + (p2 + p3);
                    }
                    __syncwarp();
                }
                __syncthreads();
                if (tid < K) run += (wsum[0][tid] + wsum[1][tid]) + (wsum[2][tid] + wsum[3][tid]);
                __syncthreads();
            }
            u += len;
        }
    }
    if (tid < K) records[(size_t)c * K + tid] = run;             // every CTA, also one without units (zeros)

    // ---- 3. grid-wide barrier, then CTA k computes output q_k ------------------------------------------------------------------
    __threadfence();
    cooperative_groups::this_grid().sync();
    const double nan = __longlong_as_double(0x7ff8000000000000LL);
    for (int k = c; k < M; k += G) {
        double s1 = 0.0, s2 = 0.0, tot = 0.0;
        for (int i = tid; i < N; i += DEBYE_IB) { const double f = (double)ff[(size_t)i * M + k]; s1 += f; s2 += f * f; }
        const int l = k + koff - 1;                                   // chain slot of q_k; -1: q_k == 0
        if (l >= 0 && l < K && U > 0)
            for (int cc = tid; cc < G; cc += DEBYE_IB) tot += __ldcg(records + (size_t)cc * K + l);
        s1 = pas_block_sum(s1, red, tid);
        s2 = pas_block_sum(s2, red, tid);
        tot = pas_block_sum(tot, red, tid);
        if (tid == 0) {
            const double qk = (double)q[k];
            out[k] = bad ? nan : ((qk == 0.0) ? s1 * s1 : s2 + tot / qk);
        }
    }
}

}  // namespace debye
