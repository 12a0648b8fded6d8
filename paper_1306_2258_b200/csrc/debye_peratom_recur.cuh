// debye_peratom_recur.cuh -- per-ATOM form factors on a uniform grid q_k = (k + koff) dq: the recurrence.
//
//     I(q_m) = sum_i ff[i][m]^2 + 2 sum_{i<j} ff[i][m] ff[j][m] sin(q_m r_ij) / (q_m r_ij)          (Eq. 2)
//
// With a different f on every atom the weights f_i f_j sit inside the pair sum, so the product form of the per-type kernel
// does not apply (its two telescoped terms would need different weights).  The CHAIN form does: per pair the three-term
// (Chebyshev) recurrence v_{m+1} = 2cos(S theta) v_m - v_{m-1} generates 2 sin(q_k r)/r for all k of the chunk (4 packed chains,
// 8 residues mod S = 8 n_chunks), and each value is accumulated with ONE packed FMA against f_j(q_k) read from shared memory:
//     acc_i[k] += f_j[k] * v[k];        at the flush  S_i[k] = f_i[k] * acc_i[k]  goes to FP64.
// 2 FP32-pipe lane-operations per term and a quarter of an LDS.128, against ~9 instructions and one MUFU.SIN per term of the
// direct kernel (debye_peratom.cuh), which stays for non-uniform and general-start grids.
//   * debye_peratom_pack_kernel: float4 positions; form factors re-laid as ffp[chunk][atom][slot] (slot order of the chains,
//     debye_pairs.cuh slot_of), pre-multiplied by the chains' sign pattern sigma_m = (+,+,-,-), padded with zeros; it also
//     classifies the q grid and records whether the caller's hint was right.
//   * debye_peratom_recur_kernel<K>: thread = one i atom of a row of 128, K accumulators; j atoms stream through shared memory
//     in tiles of DEBYE_PAR_JT atoms (position + K form factors each) by two bulk async copies per tile completing on an mbarrier,
//     double buffered.  Units (one j atom against one row) are linearised chunk -> row -> j and cut into G equal ranges.
//   * records are summed in CTA order by debye_peratom_final_kernel (mode 1: chain slots, sums of 2 sin/r).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include "debye_plan.cuh"
#include "debye_pairs.cuh"

namespace debye {

#define DEBYE_PAR_JT 64          // largest tile (the workspace is padded by one)
// j atoms per tile: JT x (16 + 4 K) bytes, two buffers, within the 48 KB of static shared memory
#ifndef DEBYE_PAR_JT_OF
#define DEBYE_PAR_JT_OF(K) ((K) <= 64 ? 64 : ((K) <= 104 ? 48 : 40))
#endif
#define DEBYE_PAR_FLUSH 512

struct PeratomPlan { int32_t bad, koff; double dq; };

// grid = (ceil(N / 256), n_chunks + 1): y < n_chunks packs chunk y of the form factors, y == n_chunks the positions (and block
// (0, n_chunks) classifies the grid).  K slots per chunk.
static __global__ void __launch_bounds__(256) debye_peratom_pack_kernel(const float *__restrict__ xyz, const float *__restrict__ ff, const float *__restrict__ q, int N, int M,
                                                                   int K, int n_chunks, int hint_class, float4 *__restrict__ pos4, float *__restrict__ ffp,
                                                                   PeratomPlan *__restrict__ plan, int B)
{
    pdl_trigger();                         // first kernel of the call: the next grids are staged while this one runs
    const int y = blockIdx.y;
    if (y == n_chunks) {
        const int64_t NB = (int64_t)N * B;                  // positions of all conformers, [B][N]
        for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < NB; i += (int64_t)gridDim.x * blockDim.x) {
            const float *s = xyz + (size_t)i * 3;
            pos4[i] = make_float4(s[0], s[1], s[2], 0.f);
        }
        if (blockIdx.x == 0) {
            __shared__ float red[8], red2[8];
            const double q0 = (double)q[0];
            const double dq = debye_grid_dq(q0, (double)q[M - 1], M);
            float dev = 0.f, qmax = 0.f;
            for (int k = threadIdx.x; k < M; k += blockDim.x) {
                const double qk = (double)q[k];
                dev = fmaxf(dev, debye_grid_dev(qk, k, q0, dq));
                qmax = fmaxf(qmax, fabsf((float)qk));
            }
            for (int o = 16; o > 0; o >>= 1) { dev = fmaxf(dev, __shfl_xor_sync(0xffffffffu, dev, o)); qmax = fmaxf(qmax, __shfl_xor_sync(0xffffffffu, qmax, o)); }
            if ((threadIdx.x & 31) == 0) { red[threadIdx.x >> 5] = dev; red2[threadIdx.x >> 5] = qmax; }
            __syncthreads();
            if (threadIdx.x == 0) {
                for (int w = 1; w < 8; ++w) { dev = fmaxf(dev, red[w]); qmax = fmaxf(qmax, red2[w]); }
                const int cls = debye_grid_class(q0, dq, dev, qmax);
                plan->koff = cls; plan->dq = dq;
                plan->bad = (cls != hint_class || cls < 0) ? 1 : 0;
            }
        }
        return;
    }
    // chunk y: slot l of atom i holds sigma_m ff[i][k], chain index idx = k + koff - 1 with slot_of(idx) = (y, l); the grid class is
    // the caller's promise here (a wrong promise is caught above and the output becomes NaN)
    const int koff = hint_class, S = 8 * n_chunks;
    const int64_t total = (int64_t)N * K;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        const int i = (int)(e / K), l = (int)(e - (int64_t)i * K);
        const int m = l >> 3, idx = S * m + 8 * y + (l & 7);          // inverse of slot_of for the recurrence
        const int k = idx + 1 - koff;
        const float v = (k >= 0 && k < M) ? ff[(size_t)i * M + k] : 0.f;
        ffp[((size_t)y * N + i) * K + l] = (m & 2) ? -v : v;
    }
}

enum PeratomMode : int { PM_C1 = 0, PM_C2A = 1, PM_C2B = 2 };

// Stage B of the chain start-up for grids q_k' = k' dq: Bv = w_0 = v(k0) for the chunk's 8 residues, A = w_{-1} = -v(k0 - S)
// = +v(S - k0) (v(-n) = -v(n), v(0) = 0), cS = 2 cos(S theta).  v_n = 2 sin(n theta)/r from the folded sine / cosine of theta/2
// and double-angle / three-term steps (one rounding each: relative accuracy survives small theta).
template <int MODE>
__device__ __forceinline__ void chain_vals(const RecurGeom &g, u64 (&A)[4], u64 (&Bv)[4], float &cS)
{
    const float rinv = g.rinv;
    cS = two_cos_from(sincos_fold(g.fS));
    const Folded h = sincos_fold(g.f1);
    const float T1 = two_sin_from(h, g.f1);
    const float c1 = two_cos_from(h);
    const float c2 = fmaf(-T1, T1, 2.0f);
    const float c4 = fmaf(c2, c2, -2.0f);
    float u[17];
    u[0] = 0.0f;
    u[1] = T1 * rinv; u[2] = c1 * u[1]; u[3] = fmaf(c1, u[2], -u[1]); u[4] = c2 * u[2];
    u[5] = fmaf(c4, u[1], u[3]); u[6] = fmaf(c4, u[2], u[2]); u[7] = fmaf(c4, u[3], u[1]); u[8] = c4 * u[4];
    if constexpr (MODE != PM_C1) {
#pragma unroll
        for (int n = 9; n <= 16; ++n) u[n] = fmaf(c4, u[n - 4], -u[n - 8]);
    }
    if constexpr (MODE == PM_C1) {
        Bv[0] = pk2(u[1], u[2]); Bv[1] = pk2(u[3], u[4]); Bv[2] = pk2(u[5], u[6]); Bv[3] = pk2(u[7], u[8]);
        A[0] = pk2(u[7], u[6]); A[1] = pk2(u[5], u[4]); A[2] = pk2(u[3], u[2]); A[3] = pk2(u[1], u[0]);
    } else if constexpr (MODE == PM_C2A) {
        Bv[0] = pk2(u[1], u[2]); Bv[1] = pk2(u[3], u[4]); Bv[2] = pk2(u[5], u[6]); Bv[3] = pk2(u[7], u[8]);
        A[0] = pk2(u[15], u[14]); A[1] = pk2(u[13], u[12]); A[2] = pk2(u[11], u[10]); A[3] = pk2(u[9], u[8]);
    } else {
        Bv[0] = pk2(u[9], u[10]); Bv[1] = pk2(u[11], u[12]); Bv[2] = pk2(u[13], u[14]); Bv[3] = pk2(u[15], u[16]);
        A[0] = pk2(u[7], u[6]); A[1] = pk2(u[5], u[4]); A[2] = pk2(u[3], u[2]); A[3] = pk2(u[1], u[0]);
    }
}

// One pair: K/8 steps of the 4 packed chains; w_m = sigma_m v_m, w_{m+1} = (+/-) cS w_m + w_{m-1}; acc[slot] += (sigma f_j)[slot] w_m.
// fj: this j atom's K pre-signed form factors in shared memory (16-byte aligned, the same address for every lane: broadcast).
template <int K>
__device__ __forceinline__ void chain_hot(u64 (&acc)[K / 2], u64 (&A)[4], u64 (&Bv)[4], const float cS, const float *__restrict__ fj)
{
    const u64 cP = pk2(cS, cS), cN = pk2(-cS, -cS);
#pragma unroll
    for (int m = 0; m < (K + 7) / 8; ++m) {
        const ulonglong2 f01 = *reinterpret_cast<const ulonglong2 *>(fj + 8 * m);              // slots 8 m .. 8 m + 3 as two pairs
        ulonglong2 f23 = f01;
        if (8 * m + 4 < K) f23 = *reinterpret_cast<const ulonglong2 *>(fj + 8 * m + 4);
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            if (8 * m + 2 * a < K) {                       // K % 8 == 4: the last step runs chains 0 and 1 only
                const u64 fp = (a == 0) ? f01.x : (a == 1) ? f01.y : (a == 2) ? f23.x : f23.y;
                acc[4 * m + a] = fma2(fp, Bv[a], acc[4 * m + a]);
                if (8 * (m + 1) + 2 * a < K) {
                    const u64 nx = fma2((m & 1) ? cN : cP, Bv[a], A[a]);
                    A[a] = Bv[a];
                    Bv[a] = nx;
                }
            }
        }
    }
}

// One tile of j atoms against this thread's i atom: the three-stage pipeline of recur_tile (stage B of pair jj + NP, stage A
// of pair jj + 2 NP, chains of pair jj), NP pairs per iteration, ONE copy of the loop per chunk mode (the mode is a template
// parameter: a run-time branch between the three start-ups inside the loop splits its basic block, and the scheduler can
// then no longer hide the start-up's dependency chains under the packed chain instructions).  Returns whether some pair of
// this thread took the small-theta mask (contributed zero; the caller rescans the tile).
// measured on B200 (T pair.q/s, cfg2 / cfg3): mode as a run-time branch inside the loop, 1 pair per iteration, 32-atom tiles
// 5.08 / 6.66; one loop per mode 5.69 / 7.62; two pairs per iteration 5.93 / 8.04; 48-atom tiles (K = 104) 6.01 / 8.17;
// 3 CTAs per SM at K = 104 (168 registers, 1 pair per iteration) 5.73 / 7.79
// two copies of the body with the roles of (A, Bv) and (An, Bn) exchanged (no register moves at the loop's tail: 55 of its 452
// instructions are MOVs): 6.00 / 7.98 against 6.19 / 8.18 (K = 104 spills 108 bytes instead of 44) -- not kept
// three pairs per iteration for K <= 64: cfg4 as a batch (K = 64) 6.58 against 6.59, 4000 atoms x 50 q (K = 56) 3.57 / 3.65 -- not kept
#ifndef DEBYE_PAR_NP
#define DEBYE_PAR_NP 2
#endif
#ifndef DEBYE_PAR_K3
#define DEBYE_PAR_K3 64          // up to this K: 3 CTAs per SM (168 registers)
#endif
template <int K, int MODE>
__device__ __forceinline__ bool peratom_tile(u64 (&acc)[K / 2], const float4 *__restrict__ tile, const float *__restrict__ tf, const int jj0, const int cnt,
                                             const float4 pi, const int jmin, const RecurConst &rc)
{
    constexpr int NP = DEBYE_PAR_NP;
    bool had_slow = false;
    auto geom = [&](const int jbase, RecurGeom (&g)[NP]) {
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            const int j = jbase + p;
            recur_geom<RM_G, false>(tile[min(j, cnt - 1)], pi, j >= jmin && j < cnt, rc, g[p]);     // RM_G: with the small-theta mask
            had_slow = had_slow || g[p].slow;
        }
    };
    u64 A[NP][4], Bv[NP][4];
    float cS[NP];
    RecurGeom gn[NP];
    geom(jj0, gn);
#pragma unroll
    for (int p = 0; p < NP; ++p) chain_vals<MODE>(gn[p], A[p], Bv[p], cS[p]);
    geom(jj0 + NP, gn);
    for (int jj = jj0; jj < cnt; jj += NP) {
        u64 An[NP][4], Bn[NP][4];
        float cSn[NP];
#pragma unroll
        for (int p = 0; p < NP; ++p) chain_vals<MODE>(gn[p], An[p], Bn[p], cSn[p]);
        geom(jj + 2 * NP, gn);
#pragma unroll
        for (int p = 0; p < NP; ++p) chain_hot<K>(acc, A[p], Bv[p], cS[p], tf + (size_t)min(jj + p, cnt - 1) * K);   // a masked pair has zero start values
#pragma unroll
        for (int p = 0; p < NP; ++p) {
#pragma unroll
            for (int a = 0; a < 4; ++a) { A[p][a] = An[p][a]; Bv[p][a] = Bn[p][a]; }
            cS[p] = cSn[p];
        }
    }
    return had_slow;
}

// BATCH: several conformers on the unit line (debye_profile_peratom_batch).  A template parameter: the kernel uses all 255
// registers at K >= 96, and the conformer's state as run-time values cost the single-structure call 4 % (spills).
template <int K, bool BATCH>
__global__ void __launch_bounds__(DEBYE_IB, K <= DEBYE_PAR_K3 ? 3 : 2) debye_peratom_recur_kernel(const float4 *__restrict__ pos4, const float *__restrict__ ffp, const float *__restrict__ qv,
                                                                                         const PeratomPlan *__restrict__ plan, int N, int M, int n_chunks, float theta_min,
                                                                                         double *__restrict__ records, int B)
{
    constexpr int JT = DEBYE_PAR_JT_OF(K), NW = DEBYE_IB / 32;
    static_assert(JT <= DEBYE_PAR_JT && JT % 2 == 0, "tile size");
    __shared__ __align__(128) float4 tpos[2][JT + DEBYE_TILE_PAD];
    __shared__ __align__(128) float tff[2][JT][K];
    __shared__ __align__(8) u64 mbar[2];
    __shared__ double wsum[NW][K];
    pdl_wait();
    if (plan->bad) return;                                  // the final kernel writes NaN
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = gridDim.x, c = blockIdx.x;
    const int rows = debye_diag_rows(N);
    const int64_t U1 = rows > 0 ? debye_diag_row_prefix(N, rows) : 0;
    const int64_t U = U1 * n_chunks * (BATCH ? B : 1);      // unit line: conformer -> chunk -> row -> j
    if (U == 0) return;
    const int64_t u0 = debye_range_begin(U, c, G);
    const int64_t u1 = (c + 1 == G) ? U : debye_range_begin(U, c + 1, G);
    if (u0 >= u1) return;

    for (int x = tid; x < 2 * (JT + DEBYE_TILE_PAD); x += DEBYE_IB) (&tpos[0][0])[x] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (tid == 0) { mbar_init(&mbar[0], 1); mbar_init(&mbar[1], 1); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();
    uint32_t phase0 = 0, phase1 = 0;

    const int S = 8 * n_chunks;
    const double dq_d = plan->dq;
    RecurConst rc;
    {
        const double w1_d = dq_d * 0.15915494309189535;
        rc.w1 = (float)w1_d; rc.w1_lo = (float)(w1_d - (double)rc.w1);
        rc.wS = rc.wS_lo = rc.w4 = rc.w4_lo = 0.f;
        rc.smult = (float)S; rc.n_chunks = n_chunks;
        const float rcut = theta_min / fabsf((float)dq_d);
        rc.cut2 = rcut * rcut;
    }
    const int koff = plan->koff;
    u64 acc[K / 2];
#pragma unroll
    for (int i = 0; i < K / 2; ++i) acc[i] = 0;
    double run = 0.0;                  // thread l < K: FP64 running sum of slot l of the current chunk
    int X_cur = -1;                    // record slot (conformer, chunk) the running sums belong to (< 65535 x 2)

    int64_t u = u0;
    while (u < u1) {
        // ---- decode unit u -> (conformer, q-chunk, row, first j) ---------------------------------------------------------
        const int X = (int)(u / U1);
        const int b = BATCH ? X / n_chunks : 0, ch = X - b * n_chunks;
        const int64_t v = u - (int64_t)X * U1;
        const int64_t boff = BATCH ? (int64_t)b * N : 0;       // this conformer's positions
        int rl = 0, rh = rows;
        while (rh - rl > 1) { const int mid = (rl + rh) >> 1; if (debye_diag_row_prefix(N, mid) <= v) rl = mid; else rh = mid; }
        const int row = rl;
        const int64_t jo = v - debye_diag_row_prefix(N, row);
        const int64_t row_units = (int64_t)N - 1 - (int64_t)row * DEBYE_IB;
        const int len = (int)min(min((int64_t)(u1 - u), row_units - jo), (int64_t)DEBYE_PAR_FLUSH);
        if (X != X_cur) {
            if (X_cur >= 0 && tid < K) { records[((int64_t)c + X_cur) * K + tid] = run; run = 0.0; }
            X_cur = X;
        }
        const int mode = (n_chunks == 1) ? PM_C1 : (ch == 0 ? PM_C2A : PM_C2B);
        const int i = row * DEBYE_IB + tid;
        const bool ivalid = i < N;
        const float4 pi = pos4[boff + (ivalid ? i : 0)];
        const int j_first = row * DEBYE_IB + 1 + (int)jo;
        const float *ffc = ffp + (size_t)ch * N * K;
        const int ntile = (len + JT - 1) / JT;

        auto issue = [&](int t, int buf) {
            const int cnt = min(len - t * JT, JT);
            const uint32_t pb = (uint32_t)cnt * 16u, fb = (uint32_t)cnt * (uint32_t)K * 4u;
            mbar_expect_tx(&mbar[buf], pb + fb);
            bulk_g2s(&tpos[buf][0], pos4 + boff + j_first + t * JT, pb, &mbar[buf]);
            bulk_g2s(&tff[buf][0][0], ffc + (size_t)(j_first + t * JT) * K, fb, &mbar[buf]);
        };
        if (tid == 0) issue(0, 0);
        for (int t = 0; t < ntile; ++t) {
            const int buf = t & 1;
            if (tid == 0 && t + 1 < ntile) issue(t + 1, buf ^ 1);
            if (buf == 0) { mbar_wait(&mbar[0], phase0); phase0 ^= 1; } else { mbar_wait(&mbar[1], phase1); phase1 ^= 1; }
            const int cnt = min(len - t * JT, JT), jl0 = j_first + t * JT;
            const float4 *tile = tpos[buf];
            // rows are diagonal blocks of the j > i triangle: a warp whose every i is >= j has nothing to do for that j
            const int jj0 = max(0, row * DEBYE_IB + warp * 32 + 1 - jl0);
            if (jj0 < cnt && row * DEBYE_IB + warp * 32 < N) {
                const int jmin = ivalid ? max(0, i + 1 - jl0) : 0x7fffffff;
                bool had_slow;
                const float *tf = &tff[buf][0][0];
                switch (mode) {      // warp-uniform; one copy of the pipelined loop per mode
                    case PM_C1: had_slow = peratom_tile<K, PM_C1>(acc, tile, tf, jj0, cnt, pi, jmin, rc); break;
                    case PM_C2A: had_slow = peratom_tile<K, PM_C2A>(acc, tile, tf, jj0, cnt, pi, jmin, rc); break;
                    default: had_slow = peratom_tile<K, PM_C2B>(acc, tile, tf, jj0, cnt, pi, jmin, rc); break;
                }
                // pairs with theta at or below theta_min (the chain would lose their frequency) and coincident atoms contributed
                // zero above; they are rare: the tile is rescanned only if some lane of the warp met one, term by term
                if (__any_sync(0xffffffffu, had_slow)) {
                    if (had_slow) {
                        for (int j = max(jj0, jmin); j < cnt; ++j) {
                            const float4 pj = tile[j];
                            const float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
                            const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                            if (!(fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, 1e-30f))) > rc.cut2)) {
                                const float rs = sqrtf(r2);
#pragma unroll
                                for (int l = 0; l < K; ++l) {
                                    const int m = l >> 3, idx = S * m + 8 * ch + (l & 7);
                                    const float qk = (float)((double)(idx + 1) * dq_d);
                                    float tv = 2.0f * ((rs == 0.0f) ? qk : term_accurate(qk, rs));     // the chains accumulate 2 sin(q r)/r
                                    if (m & 2) tv = -tv;                                                // the stored form factor carries sigma_m
                                    float lo, hi;
                                    upk2(acc[l / 2], lo, hi);
                                    if (l & 1) hi = fmaf(tff[buf][j][l], tv, hi); else lo = fmaf(tff[buf][j][l], tv, lo);
                                    acc[l / 2] = pk2(lo, hi);
                                }
                            }
                        }
                    }
                }
            }
            __syncthreads();
        }
        // ---- flush: times sigma f_i (the stored row), FP64, fixed order (xor tree over the lanes, then the warps in order) -----
        {
            const float *fi = ffc + (size_t)(ivalid ? i : 0) * K;
#pragma unroll
            for (int l = 0; l < K; l += 2) {
                float lo, hi;
                upk2(acc[l / 2], lo, hi);
                acc[l / 2] = 0;
                // (sigma f_j v)(sigma f_i) would carry sigma twice: the stored f_i row is signed too, so undo one sign
                const float s_m = ((l >> 3) & 2) ? -1.0f : 1.0f;
                double v0 = ivalid ? (double)lo * (double)(s_m * fi[l]) : 0.0, v1 = ivalid ? (double)hi * (double)(s_m * fi[l + 1]) : 0.0;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) { v0 += __shfl_xor_sync(0xffffffffu, v0, o); v1 += __shfl_xor_sync(0xffffffffu, v1, o); }
                if (lane == 0) { wsum[warp][l] = v0; wsum[warp][l + 1] = v1; }
            }
            __syncthreads();
            if (tid < K) {
                double s = 0.0;
#pragma unroll
                for (int w = 0; w < NW; ++w) s += wsum[w][tid];
                run += s;
            }
            (void)koff;
        }
        u += len;
    }
    if (X_cur >= 0 && tid < K) records[((int64_t)c + X_cur) * K + tid] = run;
}

}  // namespace debye
